// stage_kernel.cuh -- the fused SSP-RK stage kernel of the CUDA path (sm_100a, fp64).
//
// One launch performs, for a tile of TX x TY x TZ elements per thread block (one thread per nodal
// point, PAPER.md:128-145 order of operations):
//   1. stage the tile's nodal primitives W (recovered by the previous stage, Eq. 16) and the
//      one-node-deep face layer of the neighbouring elements in shared memory (with GLL nodes the
//      face interpolation of :132-134 is a gather of that layer, reading R1);
//   2. HLL interface flux (Eq. 21-24, reading R9), each face point of the tile once, spread
//      evenly over the block's threads                                          -> shared memory;
//   3. per direction: physical flux at every node (Eq. 2)                       -> shared memory,
//   4. volume quadrature (Eq. 17) + surface lift (Eq. 18), both over the diagonal mass matrix;
//   MODE_RHS stops here and writes R = L(U).  MODE_STAGE continues:
//   5. SSP-RK combine  U_out = a U0 + b (U_s + dt R)   (:147-152, reading R10), dt read from
//      device memory;
//   6. physicality-enforcing operator on the cell (Eq. 25-37), cell-local reductions in shared
//      memory;
//   7. con2prim of the new state (Eq. 16 for the next stage) and, on the step's last stage, the
//      CFL wave-speed maximum (reading R11) reduced by warp shuffles + one atomicMax per block.
// HBM traffic per node and stage: W_s 40 B (+halo, mostly L2 hits), U_s 40 B, U0 40 B (a != 0),
// U_out 40 B, W_out 40 B.
#pragma once
#include "physics.cuh"

#define DG_MODE_RHS 0
#define DG_MODE_STAGE 1
#define DG_BC_PERIODIC 0
#define DG_BC_OUTFLOW 1

typedef unsigned long long dg_ull;

__host__ __device__ constexpr int dg_ipow(int b, int e) { return e <= 0 ? 1 : b * dg_ipow(b, e - 1); }

#ifndef DG_T3N4X       // tile of the 3D p=3 kernel (tuning knob)
#define DG_T3N4X 2
#define DG_T3N4Y 2
#define DG_T3N4Z 1
#endif
// elements per thread block along x,y,z for [ndim-1][N-1]
__host__ __device__ constexpr int dg_tile(int nd, int N, int d) {
  constexpr int t[3][5][3] = {
      {{256, 1, 1}, {128, 1, 1}, {60, 1, 1}, {64, 1, 1}, {48, 1, 1}},
      {{32, 8, 1}, {16, 4, 1}, {6, 4, 1}, {4, 4, 1}, {4, 2, 1}},
      {{8, 8, 4}, {4, 4, 2}, {2, 2, 2}, {DG_T3N4X, DG_T3N4Y, DG_T3N4Z}, {2, 1, 1}}};
  return t[nd - 1][N - 1][d];
}

template <int ND, int N>
struct TileShape {
  static constexpr int NN = dg_ipow(N, ND);          // nodes per element
  static constexpr int NF1 = dg_ipow(N, ND - 1);     // nodes per element face
  static constexpr int TX = dg_tile(ND, N, 0), TY = dg_tile(ND, N, 1), TZ = dg_tile(ND, N, 2);
  static constexpr int NE = TX * TY * TZ;            // elements per tile
  static constexpr int NTN = NE * NN;                // nodes per tile
  // Threads are organised in warp groups that own whole elements, so that everything cell-local
  // (tensor-line contractions, cell mean, min s) synchronises a group, not the block:
  //   NN <= 32: one warp holds EPG = 32/NN elements (lanes >= EPG*NN idle);  NN > 32: G warps per element.
  static constexpr int G = (NN <= 32) ? 1 : (NN + 31) / 32;   // warps per group
  static constexpr int EPG = (NN <= 32) ? 32 / NN : 1;        // elements per group
  static constexpr int GT = 32 * G;                           // threads per group
  static constexpr int NG = NE / EPG;                         // groups per block
  static_assert(NE % EPG == 0, "tile must hold a whole number of warp groups");
  static_assert(G == 1 || NG <= 15, "named barriers 1..15");
  static constexpr int NT = NG * GT;                 // threads per block
  __host__ __device__ static constexpr int T(int d) { return d == 0 ? TX : (d == 1 ? TY : TZ); }
  __host__ __device__ static constexpr int SE(int d) { return d == 0 ? 1 : (d == 1 ? TX : TX * TY); }
  __host__ __device__ static constexpr int SN(int d) { return dg_ipow(N, d); }
  __host__ __device__ static constexpr int FP(int d) { return NE / T(d) * NF1; }   // points per face plane
  __host__ __device__ static constexpr int HOFF(int d) { return d <= 0 ? 0 : HOFF(d - 1) + 2 * FP(d - 1); }
  __host__ __device__ static constexpr int FOFF(int d) {
    return d <= 0 ? 0 : FOFF(d - 1) + (T(d - 1) + 1) * FP(d - 1);
  }
  static constexpr int NHALO = HOFF(ND);             // halo points of the tile
  static constexpr int NFACE = FOFF(ND);             // face points of the tile (all directions)
  // shared-memory layout, in doubles
  static constexpr int O_W = 0;                          // [5][NTN]
  static constexpr int O_F = O_W + 5 * NTN;              // [5][NTN], one direction at a time
  static constexpr int O_H = O_F + 5 * NTN;              // halo  [dir][side][5][FP]
  static constexpr int O_FH = O_H + 5 * NHALO;           // Fhat  [dir][plane][5][FP]
  static constexpr int O_D = O_FH + 5 * NFACE;           // Dhat  [N][N] (padded to 32)
  static constexpr int O_MEAN = O_D + 32;                // [NE][5]
  static constexpr int O_SMIN = O_MEAN + 5 * NE;         // [NE] (ull)
  static constexpr int O_RED = O_SMIN + NE;              // [32]
  static constexpr int O_PART = O_RED + 32;              // [NE][4][5] partial sums of the cell mean
  static constexpr int O_FLAG = O_PART + 20 * NE;        // ints: [NE] flags + [4] counters
  static constexpr int SMEM_BYTES = O_FLAG * 8 + (NE + 4) * 4 + 16;
};

struct StageArgs {
  const double* Win;      // W_s[5][ndof] primitives of the stage input state
  const double* Us;       // U_s[5][ndof]
  const double* U0;       // U at the start of the step (read only if a != 0)
  double* Uout;           // may alias Us (each thread reads and writes its own node only)
  double* Wout;           // must not alias Win
  double* Rout;           // MODE_RHS: R = L(U_s)
  long long ndof;
  int ne[3], bc[3];
  double rh[3];           // 2/h_d
  double cw[3];           // (2p+1)/h_d
  double a, b;            // Shu-Osher coefficients of this stage
  const double* dt_ptr;   // device
  double f_screen, f_solve, one_m_delta;   // 1-eps_q/2, 1-eps_q, 1-delta_s
  EosPar eos;
  dg_ull* amax;           // ordered-int image of the CFL maximum (atomicMax)
  int do_cfl;
  dg_ull* counters;       // [0] n_flagged [1] n_bad_mean [2] n_c2p_fail
  double Dhat[25];        // Dhat[i*N+q]
  double w[5];            // GLL weights
  double lift, wsum;      // 1/w_0, sum of the tensor weights (node order)
  int mode;               // DG_MODE_RHS / DG_MODE_STAGE
};

// ---------------------------------------------------------------------------------------------
// Physicality operator on a block of cells (PAPER.md:242-252 steps 1-4), one thread per node.
// Must be called by every thread of the block.  Uo: the node's state, limited in place.
//   le, n: element-in-block and node-in-element of this thread; wn: tensor GLL weight of the node.
//   scratch: >= 5*NTN doubles of shared memory free for use; sMean [NE][5]; sSmin [NE]; sFlag [NE];
//   sCnt[0..1] += flagged cells / bad means of this block.
// Returns this cell's flag; s_out receives the blend factor (1 if unflagged).
// ---------------------------------------------------------------------------------------------
template <int NN, int NE, int NTN>
__device__ __forceinline__ bool dg_limiter_block(double Uo[5], bool active, int t, int le, int n,
                                                 double wn, double wsum, double f_screen,
                                                 double f_solve, double one_m_delta,
                                                 double* scratch, double* sMean, dg_ull* sSmin,
                                                 int* sFlag, int* sCnt, double& s_out) {
  s_out = 1.0;
  bool bad = active && !dg_admissible(Uo, f_screen);               // step 1: screen (R13e)
  if (bad) sFlag[le] = 1;
  if (!__syncthreads_or(bad)) return false;                        // nothing to do in this block
  const bool flagged = active && (sFlag[le] != 0);
  if (flagged) {
#pragma unroll
    for (int v = 0; v < 5; ++v) scratch[v * NTN + t] = wn * Uo[v];
  }
  __syncthreads();
  if (flagged) {                                                   // cell average, fixed node order
    for (int v = n; v < 5; v += NN) {
      const double* p = scratch + v * NTN + le * NN;
      double acc = 0.0;
      for (int m = 0; m < NN; ++m) acc += p[m];
      sMean[le * 5 + v] = acc / wsum;
    }
  }
  __syncthreads();
  double Ub[5];
  if (flagged) {
#pragma unroll
    for (int v = 0; v < 5; ++v) Ub[v] = sMean[le * 5 + v];
    const bool mean_ok = dg_admissible(Ub, f_solve);               // step 2 (reading R13d)
    double si = 0.0;
    if (mean_ok) {
      si = dg_limiter_node_s(Ub, Uo, f_solve);                     // step 3
      if (!(si >= 0.0)) si = 0.0;
    }
    if (si < 1.0) atomicMin(&sSmin[le], dg_ord(si));               // step 4: s = min_i s_i
    if (n == 0) {
      atomicAdd(&sCnt[0], 1);
      if (!mean_ok) atomicAdd(&sCnt[1], 1);
    }
  }
  __syncthreads();
  if (flagged) {
    const double s = one_m_delta * dg_unord(sSmin[le]);            // R13c
    const double tt = 1.0 - s;
#pragma unroll
    for (int v = 0; v < 5; ++v)                                    // Eq. 26 from the nearer end (R14)
      Uo[v] = (s > 0.5) ? fma(tt, Ub[v] - Uo[v], Uo[v]) : fma(s, Uo[v] - Ub[v], Ub[v]);
    s_out = s;
  }
  return flagged;
}

// ---------------------------------------------------------------------------------------------
// helpers: decode a face point / halo point of direction D of the tile
// ---------------------------------------------------------------------------------------------
template <int ND, int N, int D>
struct DirInfo {
  using TS = TileShape<ND, N>;
  static constexpr int A = (D == 0) ? 1 : 0;        // transverse axes (ascending)
  static constexpr int B = (D == 2) ? 1 : 2;
  static constexpr int FPD = TS::FP(D);
  // transverse decode of a face-plane point fp = tn + NF1*te
  __device__ __forceinline__ static void split(int fp, int& la, int& lb, int& ca, int& cb) {
    const int te = fp / TS::NF1, tn = fp - te * TS::NF1;
    la = te % TS::T(A);
    lb = te / TS::T(A);
    ca = tn % N;
    cb = tn / N;
  }
};

// Load the halo of direction D: the facing nodal layer of the neighbouring elements (periodic wrap)
// or, at an outflow boundary, the elements' own face nodes (reading R12).  Each node on the tile's
// boundary in direction D fetches the node facing it: its global index is the thread's own index plus
// a block-uniform offset, and its halo slot is the node's face-point index.
template <int ND, int N, int D>
__device__ __forceinline__ void dg_load_halo(const StageArgs& a, double* Hs, bool active, int g,
                                             const int lc[3], const int in[3], const int org[3],
                                             const int teff[3]) {
  using TS = TileShape<ND, N>;
  using DI = DirInfo<ND, N, D>;
  constexpr int A = DI::A, B = DI::B, FPD = DI::FPD;
  int ed0 = org[D] - 1, nl0 = N - 1, ed1 = org[D] + teff[D], nl1 = 0;
  if (ed0 < 0) {
    if (a.bc[D] == DG_BC_PERIODIC) ed0 = a.ne[D] - 1;
    else { ed0 = 0; nl0 = 0; }
  }
  if (ed1 >= a.ne[D]) {
    if (a.bc[D] == DG_BC_PERIODIC) ed1 = 0;
    else { ed1 = a.ne[D] - 1; nl1 = N - 1; }
  }
  const int esD = (D == 0) ? 1 : ((D == 1) ? a.ne[0] : a.ne[0] * a.ne[1]);
  const int off0 = (ed0 - org[D]) * esD * TS::NN + nl0 * TS::SN(D);
  const int off1 = (ed1 - (org[D] + teff[D] - 1)) * esD * TS::NN + (nl1 - (N - 1)) * TS::SN(D);
  if (!active) return;
  const int fp = (in[A] + N * in[B]) + TS::NF1 * (lc[A] + TS::T(A) * lc[B]);
  double* dst = Hs + 5 * TS::HOFF(D) + fp;
  if (in[D] == 0 && lc[D] == 0) {
    const double* src = a.Win + (g + off0);
#pragma unroll
    for (int v = 0; v < 5; ++v) dst[v * FPD] = __ldg(src + v * a.ndof);
  }
  if (in[D] == N - 1 && lc[D] == teff[D] - 1) {
    const double* src = a.Win + (g + off1);
#pragma unroll
    for (int v = 0; v < 5; ++v) dst[5 * FPD + v * FPD] = __ldg(src + v * a.ndof);
  }
}

// Face point fl (0 .. (T(D)+1)*FP(D)) of direction D: pointers to the left and right face states
// (stride between variables differs for tile nodes and halo points) and to the Fhat slot.
template <int ND, int N, int D>
__device__ __forceinline__ bool dg_face_ptrs(const double* Ws, const double* Hs, double* Fh, int fl,
                                             const int teff[3], const double*& pL, int& sL,
                                             const double*& pR, int& sR, double*& pF, int& sF) {
  using TS = TileShape<ND, N>;
  using DI = DirInfo<ND, N, D>;
  constexpr int A = DI::A, B = DI::B, FPD = DI::FPD;
  const int p = fl / FPD, fp = fl - p * FPD;
  int la, lb, ca, cb;
  DI::split(fp, la, lb, ca, cb);
  if (p > teff[D] || la >= teff[A] || lb >= teff[B]) return false;
  const int tnode = ca * TS::SN(A) + cb * TS::SN(B);
  const int telem = la * TS::SE(A) + lb * TS::SE(B);
  if (p >= 1) { pL = Ws + (telem + (p - 1) * TS::SE(D)) * TS::NN + tnode + (N - 1) * TS::SN(D); sL = TS::NTN; }
  else        { pL = Hs + 5 * TS::HOFF(D) + fp; sL = FPD; }
  if (p < teff[D]) { pR = Ws + (telem + p * TS::SE(D)) * TS::NN + tnode; sR = TS::NTN; }
  else             { pR = Hs + 5 * TS::HOFF(D) + 5 * FPD + fp; sR = FPD; }
  pF = Fh + 5 * TS::FOFF(D) + p * 5 * FPD + fp;
  sF = FPD;
  return true;
}


// HLL flux at face point fl of direction D into the Fhat array.
template <int ND, int N, int EOS, int D>
__device__ __forceinline__ void dg_face_flux(const EosPar& eos, const double* Ws, const double* Hs,
                                             double* Fh, int fl, const int teff[3]) {
  const double *pL = nullptr, *pR = nullptr;
  double* pF = nullptr;
  int sL = 0, sR = 0, sF = 0;
  if (!dg_face_ptrs<ND, N, D>(Ws, Hs, Fh, fl, teff, pL, sL, pR, sR, pF, sF)) return;
  double WL[5], WR[5], F[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) { WL[v] = pL[v * sL]; WR[v] = pR[v * sR]; }
  dg_hll<EOS, D>(eos, WL, WR, F);
#pragma unroll
  for (int v = 0; v < 5; ++v) pF[v * sF] = F[v];
}

// Barrier over one warp group (G warps): __syncwarp for G = 1, else the named barrier grp+1.
template <int G>
__device__ __forceinline__ void dg_gsync(int grp) {
  if (G == 1) __syncwarp();
  else asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "r"(32 * G) : "memory");
}

// Lift of the interface flux onto a node (Eq. 18 over the diagonal mass matrix) for direction D:
//   + c * Fhat at the element's minus face if the node sits on it, - c * Fhat at its plus face,
//   c = (2/h_D) / w_0.
template <int ND, int N, int D>
__device__ __forceinline__ void dg_add_surface(const double* Fh, const int lc[3], const int in[3],
                                               double c, double R[5]) {
  using TS = TileShape<ND, N>;
  using DI = DirInfo<ND, N, D>;
  constexpr int A = DI::A, B = DI::B, FPD = DI::FPD;
  if (in[D] != 0 && in[D] != N - 1) return;
  const int fp = (in[A] + N * in[B]) + TS::NF1 * (lc[A] + TS::T(A) * lc[B]);
  const double* base = Fh + 5 * TS::FOFF(D) + fp;
  if (in[D] == 0) {
    const double* p = base + lc[D] * 5 * FPD;
#pragma unroll
    for (int v = 0; v < 5; ++v) R[v] = fma(c, p[v * FPD], R[v]);
  }
  if (in[D] == N - 1) {
    const double* p = base + (lc[D] + 1) * 5 * FPD;
#pragma unroll
    for (int v = 0; v < 5; ++v) R[v] = fma(-c, p[v * FPD], R[v]);
  }
}

// One direction of the volume term for this thread's node: flux (Eq. 2) of the node into the
// shared buffer Fb, group barrier, tensor-line contraction with Dhat (Eq. 17).  The caller
// alternates Fb between two buffers, so no barrier is needed after the reads.
template <int ND, int N, int D>
__device__ __forceinline__ void dg_direction(const StageArgs& a, const double* sD, double* Fb, int ti,
                                             bool active, int grp, const int in[3], const double Un[5],
                                             double P, double vd, double R[5]) {
  using TS = TileShape<ND, N>;
  constexpr int NTN = TS::NTN;
  if (active) {
    Fb[0 * NTN + ti] = Un[0] * vd;
    Fb[1 * NTN + ti] = fma(Un[1], vd, (D == 0) ? P : 0.0);
    Fb[2 * NTN + ti] = fma(Un[2], vd, (D == 1) ? P : 0.0);
    Fb[3 * NTN + ti] = fma(Un[3], vd, (D == 2) ? P : 0.0);
    Fb[4 * NTN + ti] = (Un[4] + P) * vd;
  }
  dg_gsync<TS::G>(grp);
  if (active) {
    const int id = in[D];
    const double* line = Fb + (ti - id * TS::SN(D));
    const double* dh = sD + id * N;
    double dq[N];
#pragma unroll
    for (int q = 0; q < N; ++q) dq[q] = a.rh[D] * dh[q];
#pragma unroll
    for (int v = 0; v < 5; ++v) {
#pragma unroll
      for (int q = 0; q < N; ++q) R[v] = fma(dq[q], line[v * NTN + q * TS::SN(D)], R[v]);
    }
  }
}

// Physicality operator on the cells of one warp group (PAPER.md:242-252 steps 1-4), one thread per
// node; cell-local reductions through shared memory with group barriers only.  Must be called by
// every thread of the group.  Uo: the node's state, limited in place.
template <int ND, int N>
__device__ __forceinline__ void dg_limiter_group(double Uo[5], bool active, int ti, int le, int n, int grp,
                                                 double wn, const StageArgs& a, double* scratch,
                                                 double* sPart, double* sMean, dg_ull* sSmin, int* sFlag,
                                                 int* sCnt) {
  using TS = TileShape<ND, N>;
  constexpr int NN = TS::NN, NTN = TS::NTN;
  const bool bad = active && !dg_admissible(Uo, a.f_screen);         // step 1: screen (R13e)
  if (bad) sFlag[le] = 1;
  dg_gsync<TS::G>(grp);
  const bool flagged = active && (sFlag[le] != 0);
  // nothing flagged in this warp group (the common case): done, no further group barriers
  const bool any = (TS::G == 1) ? (__any_sync(0xffffffffu, flagged) != 0) : (sFlag[grp * TS::EPG] != 0);
  if (!any) return;
  if (flagged) {
#pragma unroll
    for (int v = 0; v < 5; ++v) scratch[v * NTN + ti] = wn * Uo[v];
  }
  dg_gsync<TS::G>(grp);
  // cell average: J interleaved partial sums per variable (5 J lanes), then their sum by 5 lanes
  constexpr int J = (NN >= 20) ? 4 : NN / 5;
  if (J == 0) {                                                     // tiny cells: one lane sums
    if (flagged && n == 0) {
      for (int v = 0; v < 5; ++v) {
        double acc = 0.0;
        for (int m = 0; m < NN; ++m) acc += scratch[v * NTN + le * NN + m];
        sMean[le * 5 + v] = acc / a.wsum;
      }
    }
  } else {
    if (flagged && n < 5 * J) {
      const int v = n % 5, j = n / 5;
      const double* p = scratch + v * NTN + le * NN;
      double acc = 0.0;
      for (int m = j; m < NN; m += J) acc += p[m];
      sPart[le * 20 + n] = acc;
    }
    dg_gsync<TS::G>(grp);
    if (flagged && n < 5) {
      double acc = 0.0;
#pragma unroll
      for (int j = 0; j < J; ++j) acc += sPart[le * 20 + 5 * j + n];
      sMean[le * 5 + n] = acc / a.wsum;
    }
  }
  dg_gsync<TS::G>(grp);
  double Ub[5];
  if (flagged) {
#pragma unroll
    for (int v = 0; v < 5; ++v) Ub[v] = sMean[le * 5 + v];
    const bool mean_ok = dg_admissible(Ub, a.f_solve);               // step 2 (reading R13d)
    double si = 0.0;
    if (mean_ok) {
      si = dg_limiter_node_s(Ub, Uo, a.f_solve);                     // step 3
      if (!(si >= 0.0)) si = 0.0;
    }
    if (si < 1.0) atomicMin(&sSmin[le], dg_ord(si));                 // step 4: s = min_i s_i
    if (n == 0) {
      atomicAdd(&sCnt[0], 1);
      if (!mean_ok) atomicAdd(&sCnt[1], 1);
    }
  }
  dg_gsync<TS::G>(grp);
  if (flagged) {
    const double s = a.one_m_delta * dg_unord(sSmin[le]);            // R13c
    const double tt = 1.0 - s;
#pragma unroll
    for (int v = 0; v < 5; ++v)                                      // Eq. 26 from the nearer end (R14)
      Uo[v] = (s > 0.5) ? fma(tt, Ub[v] - Uo[v], Uo[v]) : fma(s, Uo[v] - Ub[v], Ub[v]);
  }
}

// resident blocks per SM the register allocation must allow: 1024 threads (32 warps) per SM
#ifndef DG_MINB
#define DG_MINB (1024 / TileShape<ND, N>::NT)
#endif
template <int ND, int N, int EOS>
__global__ void __launch_bounds__(TileShape<ND, N>::NT, DG_MINB)
dg_stage_kernel(const __grid_constant__ StageArgs a) {
  using TS = TileShape<ND, N>;
  constexpr int NN = TS::NN, NTN = TS::NTN, NT = TS::NT, NE = TS::NE;
  extern __shared__ __align__(16) double sm[];
  double* Ws = sm + TS::O_W;
  double* Fs = sm + TS::O_F;
  double* Hs = sm + TS::O_H;
  double* Fh = sm + TS::O_FH;
  double* sD = sm + TS::O_D;
  double* sMean = sm + TS::O_MEAN;
  dg_ull* sSmin = reinterpret_cast<dg_ull*>(sm + TS::O_SMIN);
  double* sRed = sm + TS::O_RED;
  double* sPart = sm + TS::O_PART;
  int* sFlag = reinterpret_cast<int*>(sm + TS::O_FLAG);
  int* sCnt = sFlag + NE;

  // tile of this block
  const int org[3] = {(int)blockIdx.x * TS::TX, (int)blockIdx.y * TS::TY, (int)blockIdx.z * TS::TZ};
  const int teff[3] = {min(TS::TX, a.ne[0] - org[0]), min(TS::TY, a.ne[1] - org[1]),
                       min(TS::TZ, a.ne[2] - org[2])};
  // warp group, element and node of this thread
  const int t = threadIdx.x;
  const int grp = t / TS::GT, r = t - grp * TS::GT;
  const int le = grp * TS::EPG + r / NN, n = r % NN;
  const int ti = le * NN + n;                                        // node slot in the tile arrays
  const int lc[3] = {le % TS::TX, (le / TS::TX) % TS::TY, le / (TS::TX * TS::TY)};
  const int in[3] = {n % N, (n / N) % N, n / (N * N)};
  const bool active = (r < TS::EPG * NN) && lc[0] < teff[0] && lc[1] < teff[1] && lc[2] < teff[2];
  int g = 0;                                                         // ndof < 2^31 (dgrhd_create)
  if (active) g = ((org[0] + lc[0]) + a.ne[0] * ((org[1] + lc[1]) + a.ne[1] * (org[2] + lc[2]))) * NN + n;
  if (t < NE) { sSmin[t] = dg_ord(1.0); sFlag[t] = 0; }
  if (t < 4) sCnt[t] = 0;
  if (t < N * N) sD[t] = a.Dhat[t];

  // 1. stage W of the tile and of the neighbours' facing nodal layers; U_s of the node in flight
  double P = 1.0, v0 = 0.0, v1 = 0.0, v2 = 0.0, Un[5] = {0, 0, 0, 0, 0};
  if (active) {
    double Wn[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      Wn[v] = __ldg(a.Win + v * a.ndof + g);
      Ws[v * NTN + ti] = Wn[v];
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) Un[v] = a.Us[v * a.ndof + g];
    const double rg = dg_rsqrt(fma(Wn[1], Wn[1], fma(Wn[2], Wn[2], fma(Wn[3], Wn[3], 1.0))));
    P = Wn[4]; v0 = Wn[1] * rg; v1 = Wn[2] * rg; v2 = Wn[3] * rg;
  }
  dg_load_halo<ND, N, 0>(a, Hs, active, g, lc, in, org, teff);
  if constexpr (ND > 1) dg_load_halo<ND, N, 1>(a, Hs, active, g, lc, in, org, teff);
  if constexpr (ND > 2) dg_load_halo<ND, N, 2>(a, Hs, active, g, lc, in, org, teff);
  __syncthreads();

  // 2. interface flux at every face point of the tile, once each, spread over all threads
  for (int f = t; f < TS::NFACE; f += NT) {
    if (ND == 1 || f < TS::FOFF(1)) dg_face_flux<ND, N, EOS, 0>(a.eos, Ws, Hs, Fh, f, teff);
    else if (ND == 2 || f < TS::FOFF(2)) dg_face_flux<ND, N, EOS, (ND > 1 ? 1 : 0)>(a.eos, Ws, Hs, Fh, f - TS::FOFF(1), teff);
    else dg_face_flux<ND, N, EOS, (ND > 2 ? 2 : 0)>(a.eos, Ws, Hs, Fh, f - TS::FOFF(2), teff);
  }

  // 3. volume quadrature, direction by direction, F(W_i) = U_i v_d + P e_d; the first direction
  //    overlaps other warps' face fluxes, the block barrier then frees Ws as the second F buffer
  double R[5] = {0, 0, 0, 0, 0};
  dg_direction<ND, N, 0>(a, sD, Fs, ti, active, grp, in, Un, P, v0, R);
  __syncthreads();
  if constexpr (ND > 1) dg_direction<ND, N, 1>(a, sD, Ws, ti, active, grp, in, Un, P, v1, R);
  if constexpr (ND > 2) dg_direction<ND, N, 2>(a, sD, Fs, ti, active, grp, in, Un, P, v2, R);

  // 4. surface lift
  if (active) {
    dg_add_surface<ND, N, 0>(Fh, lc, in, a.rh[0] * a.lift, R);
    if constexpr (ND > 1) dg_add_surface<ND, N, 1>(Fh, lc, in, a.rh[1] * a.lift, R);
    if constexpr (ND > 2) dg_add_surface<ND, N, 2>(Fh, lc, in, a.rh[2] * a.lift, R);
  }
  if (a.mode == DG_MODE_RHS) {
    if (active) {
#pragma unroll
      for (int v = 0; v < 5; ++v) a.Rout[v * a.ndof + g] = R[v];
    }
    return;
  }

  // 5. SSP-RK combine (Shu-Osher form)
  const double dt = *a.dt_ptr;
  double Uo[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) Uo[v] = a.b * fma(dt, R[v], Un[v]);
  if (a.a != 0.0 && active) {
#pragma unroll
    for (int v = 0; v < 5; ++v) Uo[v] = fma(a.a, a.U0[v * a.ndof + g], Uo[v]);
  }

  // 6. physicality-enforcing operator (cell-local)
  double wn = a.w[in[0]];
  if (ND > 1) wn *= a.w[in[1]];
  if (ND > 2) wn *= a.w[in[2]];
  dg_limiter_group<ND, N>(Uo, active, ti, le, n, grp, wn, a, (ND == 2) ? Fs : Ws, sPart, sMean, sSmin,
                          sFlag, sCnt);

  // 7. primitives of the new state, CFL maximum
  double speed = 0.0;
  if (active) {
    double Wo[5];
    const int st = dg_con2prim<EOS>(a.eos, Uo, Wo);
    if (st != 0) atomicAdd(&sCnt[2], 1);
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      a.Uout[v * a.ndof + g] = Uo[v];
      a.Wout[v * a.ndof + g] = Wo[v];
    }
    if (a.do_cfl) {
      const double sp = dg_cfl_speed<EOS, ND>(a.eos, Wo, a.cw);
      if (sp > 0.0) speed = sp;
    }
  }
  if (a.do_cfl) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) speed = fmax(speed, __shfl_xor_sync(0xffffffffu, speed, o));
    if ((t & 31) == 0) sRed[t >> 5] = speed;
  }
  __syncthreads();
  if (t < 32) {
    if (a.do_cfl) {
      double y = (t < NT / 32) ? sRed[t] : 0.0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) y = fmax(y, __shfl_xor_sync(0xffffffffu, y, o));
      if (t == 0 && y > 0.0) atomicMax(a.amax, dg_ord(y));
    }
    if (t < 3 && sCnt[t]) atomicAdd(&a.counters[t], (dg_ull)sCnt[t]);
  }
}

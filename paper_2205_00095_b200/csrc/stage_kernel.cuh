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

#ifndef DG_T3N4
#define DG_T3N4 2, 2, 2
#endif
// elements per thread block along x,y,z for [ndim-1][N-1]
__host__ __device__ constexpr int dg_tile(int nd, int N, int d) {
  constexpr int t[3][5][3] = {
      {{256, 1, 1}, {128, 1, 1}, {64, 1, 1}, {64, 1, 1}, {48, 1, 1}},
      {{32, 8, 1}, {16, 4, 1}, {8, 4, 1}, {4, 4, 1}, {4, 2, 1}},
      {{8, 8, 4}, {4, 4, 2}, {4, 2, 2}, {DG_T3N4}, {2, 1, 1}}};
  return t[nd - 1][N - 1][d];
}

template <int ND, int N>
struct TileShape {
  static constexpr int NN = dg_ipow(N, ND);          // nodes per element
  static constexpr int NF1 = dg_ipow(N, ND - 1);     // nodes per element face
  static constexpr int TX = dg_tile(ND, N, 0), TY = dg_tile(ND, N, 1), TZ = dg_tile(ND, N, 2);
  static constexpr int NE = TX * TY * TZ;            // elements per tile
  static constexpr int NTN = NE * NN;                // nodes per tile
  static constexpr int NT = (NTN + 31) / 32 * 32;    // threads per block
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
  static constexpr int O_FLAG = O_RED + 32;              // ints: [NE] flags + [4] counters
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

// Load the halo point hl (0 .. 2*FP(D)) of direction D: the facing nodal layer of the neighbouring
// element (periodic wrap) or, at an outflow boundary, the element's own face node (reading R12).
template <int ND, int N, int D>
__device__ __forceinline__ void dg_load_halo(const StageArgs& a, double* Hs, int hl, const int org[3],
                                             const int teff[3]) {
  using TS = TileShape<ND, N>;
  using DI = DirInfo<ND, N, D>;
  constexpr int A = DI::A, B = DI::B, FPD = DI::FPD;
  const int side = hl / FPD, fp = hl - side * FPD;
  int la, lb, ca, cb;
  DI::split(fp, la, lb, ca, cb);
  if (la >= teff[A] || lb >= teff[B]) return;
  int ed, nd_;
  if (side == 0) {
    ed = org[D] - 1; nd_ = N - 1;
    if (ed < 0) {
      if (a.bc[D] == DG_BC_PERIODIC) ed = a.ne[D] - 1;
      else { ed = 0; nd_ = 0; }
    }
  } else {
    ed = org[D] + teff[D]; nd_ = 0;
    if (ed >= a.ne[D]) {
      if (a.bc[D] == DG_BC_PERIODIC) ed = 0;
      else { ed = a.ne[D] - 1; nd_ = N - 1; }
    }
  }
  int ec[3];
  ec[D] = ed; ec[A] = org[A] + la; ec[B] = org[B] + lb;
  const long long e = ec[0] + (long long)a.ne[0] * (ec[1] + (long long)a.ne[1] * ec[2]);
  const int n = nd_ * TS::SN(D) + ca * TS::SN(A) + cb * TS::SN(B);
  const long long g = e * TS::NN + n;
  double* dst = Hs + 5 * TS::HOFF(D) + side * 5 * FPD + fp;
#pragma unroll
  for (int v = 0; v < 5; ++v) dst[v * FPD] = __ldg(a.Win + v * a.ndof + g);
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

// Lift of the interface flux onto a node (Eq. 18 over the diagonal mass matrix) for direction D:
//   + lift * Fhat at the element's minus face if the node sits on it, - lift * Fhat at its plus face.
template <int ND, int N, int D>
__device__ __forceinline__ void dg_add_surface(const double* Fh, const int lc[3], const int in[3],
                                               double lift, double acc[5]) {
  using TS = TileShape<ND, N>;
  using DI = DirInfo<ND, N, D>;
  constexpr int A = DI::A, B = DI::B, FPD = DI::FPD;
  const int fp = (in[A] + N * in[B]) + TS::NF1 * (lc[A] + TS::T(A) * lc[B]);
  const double* base = Fh + 5 * TS::FOFF(D) + fp;
  if (in[D] == 0) {
    const double* p = base + lc[D] * 5 * FPD;
#pragma unroll
    for (int v = 0; v < 5; ++v) acc[v] = fma(lift, p[v * FPD], acc[v]);
  }
  if (in[D] == N - 1) {
    const double* p = base + (lc[D] + 1) * 5 * FPD;
#pragma unroll
    for (int v = 0; v < 5; ++v) acc[v] = fma(-lift, p[v * FPD], acc[v]);
  }
}

// One direction of the spatial operator for this thread's node: flux (Eq. 2) of the node into shared
// memory, then the tensor-line contraction with Dhat (Eq. 17) and the surface lift (Eq. 18).
template <int ND, int N, int D>
__device__ __forceinline__ void dg_direction(const StageArgs& a, const double* sD, double* Fs,
                                             const double* Fh, int t, bool active, const int lc[3],
                                             const int in[3], const double Un[5], double P, double vd,
                                             double R[5]) {
  using TS = TileShape<ND, N>;
  constexpr int NTN = TS::NTN;
  if (D > 0) __syncthreads();                                    // previous direction's reads done
  if (active) {
    Fs[0 * NTN + t] = Un[0] * vd;
    Fs[1 * NTN + t] = fma(Un[1], vd, (D == 0) ? P : 0.0);
    Fs[2 * NTN + t] = fma(Un[2], vd, (D == 1) ? P : 0.0);
    Fs[3 * NTN + t] = fma(Un[3], vd, (D == 2) ? P : 0.0);
    Fs[4 * NTN + t] = (Un[4] + P) * vd;
  }
  __syncthreads();
  if (active) {
    const int id = in[D];
    const double* line = Fs + (t - id * TS::SN(D));
    const double* dh = sD + id * N;
    double acc[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      double s = 0.0;
#pragma unroll
      for (int q = 0; q < N; ++q) s = fma(dh[q], line[v * NTN + q * TS::SN(D)], s);
      acc[v] = s;
    }
    dg_add_surface<ND, N, D>(Fh, lc, in, a.lift, acc);
#pragma unroll
    for (int v = 0; v < 5; ++v) R[v] = fma(a.rh[D], acc[v], R[v]);
  }
}

template <int ND, int N, int EOS>
__global__ void __launch_bounds__(TileShape<ND, N>::NT)
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
  int* sFlag = reinterpret_cast<int*>(sm + TS::O_FLAG);
  int* sCnt = sFlag + NE;

  // tile of this block
  const int ntx = (a.ne[0] + TS::TX - 1) / TS::TX, nty = (a.ne[1] + TS::TY - 1) / TS::TY;
  const int bt = blockIdx.x;
  const int org[3] = {(bt % ntx) * TS::TX, ((bt / ntx) % nty) * TS::TY, (bt / (ntx * nty)) * TS::TZ};
  const int teff[3] = {min(TS::TX, a.ne[0] - org[0]), min(TS::TY, a.ne[1] - org[1]),
                       min(TS::TZ, a.ne[2] - org[2])};
  // node of this thread
  const int t = threadIdx.x;
  const int le = t / NN, n = t - le * NN;
  const int lc[3] = {le % TS::TX, (le / TS::TX) % TS::TY, le / (TS::TX * TS::TY)};
  const int in[3] = {n % N, (n / N) % N, n / (N * N)};
  const bool active = (t < NTN) && lc[0] < teff[0] && lc[1] < teff[1] && lc[2] < teff[2];
  long long g = 0;
  if (active) {
    const long long e = (org[0] + lc[0]) +
                        (long long)a.ne[0] * ((org[1] + lc[1]) + (long long)a.ne[1] * (org[2] + lc[2]));
    g = e * NN + n;
  }
  if (t < NE) { sSmin[t] = dg_ord(1.0); sFlag[t] = 0; }
  if (t < 4) sCnt[t] = 0;
  if (t < N * N) sD[t] = a.Dhat[t];

  // 1. stage W of the tile and of the neighbours' facing nodal layers
  double Wn[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, Un[5] = {0, 0, 0, 0, 0};
  if (active) {
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      Wn[v] = __ldg(a.Win + v * a.ndof + g);
      Ws[v * NTN + t] = Wn[v];
      Un[v] = a.Us[v * a.ndof + g];
    }
  }
  for (int hl = t; hl < 2 * TS::FP(0); hl += NT) dg_load_halo<ND, N, 0>(a, Hs, hl, org, teff);
  if constexpr (ND > 1)
    for (int hl = t; hl < 2 * TS::FP(1); hl += NT) dg_load_halo<ND, N, 1>(a, Hs, hl, org, teff);
  if constexpr (ND > 2)
    for (int hl = t; hl < 2 * TS::FP(2); hl += NT) dg_load_halo<ND, N, 2>(a, Hs, hl, org, teff);
  __syncthreads();

  // 2. interface flux at every face point of the tile, once each
  for (int f = t; f < TS::NFACE; f += NT) {
    const double *pL = nullptr, *pR = nullptr;
    double* pF = nullptr;
    int sL = 0, sR = 0, sF = 0, dir = 0;
    bool ok;
    if (ND == 1 || f < TS::FOFF(1)) {
      dir = 0; ok = dg_face_ptrs<ND, N, 0>(Ws, Hs, Fh, f, teff, pL, sL, pR, sR, pF, sF);
    } else if (ND == 2 || f < TS::FOFF(2)) {
      dir = 1; ok = dg_face_ptrs<ND, N, (ND > 1 ? 1 : 0)>(Ws, Hs, Fh, f - TS::FOFF(1), teff, pL, sL, pR, sR, pF, sF);
    } else {
      dir = 2; ok = dg_face_ptrs<ND, N, (ND > 2 ? 2 : 0)>(Ws, Hs, Fh, f - TS::FOFF(2), teff, pL, sL, pR, sR, pF, sF);
    }
    if (ok) {
      double WL[5], WR[5], F[5];
#pragma unroll
      for (int v = 0; v < 5; ++v) { WL[v] = pL[v * sL]; WR[v] = pR[v * sR]; }
      dg_hll<EOS>(a.eos, WL, WR, dir, F);
#pragma unroll
      for (int v = 0; v < 5; ++v) pF[v * sF] = F[v];
    }
  }
  __syncthreads();

  // 3.-4. volume quadrature + surface lift, one direction at a time; F(W_i) = U_i v_d + P e_d
  double R[5] = {0, 0, 0, 0, 0};
  {
    const double rg = rsqrt(fma(Wn[1], Wn[1], fma(Wn[2], Wn[2], fma(Wn[3], Wn[3], 1.0))));
    dg_direction<ND, N, 0>(a, sD, Fs, Fh, t, active, lc, in, Un, Wn[4], Wn[1] * rg, R);
    if constexpr (ND > 1) dg_direction<ND, N, 1>(a, sD, Fs, Fh, t, active, lc, in, Un, Wn[4], Wn[2] * rg, R);
    if constexpr (ND > 2) dg_direction<ND, N, 2>(a, sD, Fs, Fh, t, active, lc, in, Un, Wn[4], Wn[3] * rg, R);
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
  double s_cell;
  dg_limiter_block<NN, NE, NTN>(Uo, active, t, le, n, wn, a.wsum, a.f_screen, a.f_solve, a.one_m_delta,
                                Fs, sMean, sSmin, sFlag, sCnt, s_cell);

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

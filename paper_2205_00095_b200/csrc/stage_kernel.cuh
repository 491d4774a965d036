// stage_kernel.cuh -- the fused SSP-RK stage kernel of the CUDA path (sm_100a, fp64).
//
// One launch performs, for a tile of TX x TY x TZ elements per thread block (one thread per nodal
// point, PAPER.md:128-145 order of operations):
//   1. stage the tile's nodal primitives W (recovered by the previous stage, Eq. 16) and the
//      one-node-deep face layer of the neighbouring elements in shared memory (with GLL nodes the
//      face interpolation of :132-134 is a gather of that layer, reading R1);
//   2. physical flux at every node, every direction (Eq. 2)                      -> shared memory;
//   3. HLL interface flux (Eq. 21-24, reading R9), each face point of the tile once, spread
//      evenly over the block's threads                                          -> shared memory;
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
  static constexpr int O_F = O_W + 5 * NTN;              // [ND][5][NTN]
  static constexpr int O_H = O_F + ND * 5 * NTN;         // halo  [dir][side][5][FP]
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
  double lift, inv_wsum;  // 1/w_0, 1/sum of tensor weights
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
                                                 double wn, double inv_wsum, double f_screen,
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
      sMean[le * 5 + v] = acc * inv_wsum;
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
                                             const double*& pR, int& sR, double*& pF) {
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
  return true;
}

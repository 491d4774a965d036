// stage_kernel.cuh -- the fused SSP-RK stage kernel of the CUDA path (sm_100a, fp64).
//
// One launch performs, for a tile of TX x TY x TZ elements per thread block (one thread per nodal
// point, PAPER.md:128-145 order of operations):
//   1. per tile node a record in shared memory -- conserved state U_s, 3-velocity, pressure and the
//      fraction sigma_s = num/den of Eq. 22 -- from the node's primitives W (recovered by the previous
//      stage, Eq. 16) and U_s; the primitives of the one-node-deep face layer of the neighbouring
//      elements arrive by cp.async (with GLL nodes the face interpolation of :132-134 is a gather
//      of that layer, reading R1) and get their records (U by Eq. 4) in a dense pass;
//   2. HLL interface flux (Eq. 21-24, reading R9) from the two records of each face point of the
//      tile, once each, spread evenly over the block's threads                  -> shared memory;
//   3. volume quadrature (Eq. 17) over the diagonal mass matrix, F_d = U v_d + P e_d (Eq. 2) formed on
//      the fly from the records along the node's tensor lines (read-only: no barrier);
//   4. surface lift (Eq. 18);
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

#ifndef DG_NPT64       // nodes per thread of the 3D p=3 kernel (1 or 2)
#define DG_NPT64 1
#endif
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
  // A thread owns M nodes of one element (node n0 + m NNT, m < M): M = 2 for the 64-node hexahedron, so
  // that an element is exactly one warp (no cross-warp barrier for anything cell-local) and every
  // thread carries two independent fp64 instruction streams; M = 1 otherwise.
  static constexpr int M = (NN == 64) ? DG_NPT64 : 1;
  static constexpr int NNT = NN / M;                 // threads per element
  // Threads are organised in warp groups that own whole elements, so that everything cell-local
  // (cell mean, min s) synchronises a group, not the block:
  //   NNT <= 32: one warp holds EPG = 32/NNT elements (lanes >= EPG*NNT idle);  else G warps per element.
  static constexpr int G = (NNT <= 32) ? 1 : (NNT + 31) / 32;   // warps per group
  static constexpr int EPG = (NNT <= 32) ? 32 / NNT : 1;        // elements per group
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
  // shared-memory layout, in doubles.  Node records: per tile node X[11][NTN] = D Mx My Mz E | vx vy
  // vz | P | num den (conserved state, 3-velocity, pressure, sigma = num/den of Eq. 22); per halo
  // point XH[9][NHALO] = D Mx My Mz E | v_normal | P | num den.
  static constexpr int NREC = 11, HREC = 9;
  static constexpr int O_X = 0;                          // [NREC][NTN]
  static constexpr int O_XH = O_X + NREC * NTN;          // [HREC][NHALO]
  static constexpr int O_FH = O_XH + HREC * NHALO;       // Fhat  [dir][plane][5][FP]
  static constexpr int O_D = O_FH + 5 * NFACE;           // Dhat  [N][N] (padded to 32)
  static constexpr int O_MEAN = O_D + 32;                // [NE][5]
  static constexpr int O_SMIN = O_MEAN + 5 * NE;         // [NE] (ull)
  static constexpr int O_RED = O_SMIN + NE;              // [32]
  static constexpr int O_PART = O_RED + 32;              // [NE][4][5] partial sums of the cell mean
  static constexpr int O_FLAG = O_PART + 20 * NE;        // ints: [NE] flags + [4] counters
  static constexpr int SMEM_BYTES = O_FLAG * 8 + (NE + 4) * 4 + 16;
  static constexpr int BLK_SMEM = (227 * 1024) / (SMEM_BYTES + 1024);
  static constexpr int BLK_THR = 1024 / NT;
  static constexpr int MINB = (BLK_SMEM < BLK_THR ? BLK_SMEM : BLK_THR) > 0 ? (BLK_SMEM < BLK_THR ? BLK_SMEM : BLK_THR) : 1;
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
  int hoff[3][2], hfix[3][2];   // halo: global-index offset of the facing node (minus, plus side)
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

// Record of a tile node in the shared node array from its primitives W and conserved state U: U (for
// the Riemann flux and the volume flux F_d = U v_d + P e_d), the 3-velocity v = u/gamma, P, and
// sigma_s = num/den of Eq. 22 as an unevaluated fraction.
template <int ND, int N, int EOS>
__device__ __forceinline__ void dg_node_record(const EosPar& eos, const double W[5], const double U[5],
                                               double* X, int slot) {
  constexpr int S = TileShape<ND, N>::NTN;
  const double g2 = fma(W[1], W[1], fma(W[2], W[2], fma(W[3], W[3], 1.0)));
  const double rg = dg_rsqrt(g2);
  double num, den;
  dg_sigma_frac<EOS>(eos, W[0], W[4], g2, num, den);
  double* x = X + slot;
#pragma unroll
  for (int v = 0; v < 5; ++v) x[v * S] = U[v];
  x[5 * S] = W[1] * rg;
  x[6 * S] = W[2] * rg;
  x[7 * S] = W[3] * rg;
  x[8 * S] = W[4];
  x[9 * S] = num;
  x[10 * S] = den;
}

// Record of halo point h: its primitives W sit in rows 0..4 of XH; replace them by U (Eq. 4, reading
// R8) and add the velocity component normal to the face, P and the sigma fraction.
template <int ND, int N, int EOS>
__device__ __forceinline__ void dg_halo_record(const EosPar& eos, double* XH, int h) {
  using TS = TileShape<ND, N>;
  constexpr int S = TS::NHALO;
  double* x = XH + h;
  double W[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) W[v] = x[v * S];
  const int D = (ND > 2 && h >= TS::HOFF(2)) ? 2 : ((ND > 1 && h >= TS::HOFF(1)) ? 1 : 0);
  const double g2 = fma(W[1], W[1], fma(W[2], W[2], fma(W[3], W[3], 1.0)));
  const double rg = dg_rsqrt(g2);
  double num, den;
  dg_sigma_frac<EOS>(eos, W[0], W[4], g2, num, den);
  const double rh = dg_rho_h<EOS>(eos, W[0], W[4]);
  const double g = g2 * rg, grh = g * rh;
  x[0] = g * W[0];
  x[1 * S] = grh * W[1];
  x[2 * S] = grh * W[2];
  x[3 * S] = grh * W[3];
  x[4 * S] = fma(g2, rh, -W[4]);
  x[5 * S] = ((D == 0) ? W[1] : ((D == 1) ? W[2] : W[3])) * rg;
  x[6 * S] = W[4];
  x[7 * S] = num;
  x[8 * S] = den;
}

__device__ __forceinline__ void dg_async_copy8(double* smem_dst, const double* gmem_src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)),
               "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void dg_async_wait() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Halo of direction D: each node on the tile's boundary in direction D fetches the primitives of the
// node facing it in the neighbouring element (periodic wrap; at an outflow boundary its own, reading
// R12) -- global index = own index + a block-uniform offset -- into the halo slot that equals the
// node's face-point index (rows 0..4; the record is completed in a dense pass over the halo slots).
template <int ND, int N, int D>
__device__ __forceinline__ void dg_load_halo(const StageArgs& a, double* XH, bool active, int g,
                                             const int lc[3], const int in[3], const int org[3],
                                             const int teff[3]) {
  using TS = TileShape<ND, N>;
  using DI = DirInfo<ND, N, D>;
  constexpr int A = DI::A, B = DI::B, FPD = DI::FPD;
  // offsets of the facing node: interior value + a correction on the first / last tile of the axis
  // (periodic wrap or outflow), both precomputed by the host (StageArgs::hoff, hfix)
  const int off0 = a.hoff[D][0] + ((org[D] == 0) ? a.hfix[D][0] : 0);
  const int off1 = a.hoff[D][1] + ((org[D] + teff[D] == a.ne[D]) ? a.hfix[D][1] : 0);
  if (!active) return;
  const int fp = (in[A] + N * in[B]) + TS::NF1 * (lc[A] + TS::T(A) * lc[B]);
  double* dst = XH + (TS::HOFF(D) + fp);
  // asynchronous 8-byte copies global -> shared (LDGSTS): all halo rows of the block are in flight at
  // once and no register is held; the caller waits with dg_async_wait() before the block barrier
  if (in[D] == 0 && lc[D] == 0) {
    const double* src = a.Win + (g + off0);
#pragma unroll
    for (int v = 0; v < 5; ++v) dg_async_copy8(dst + v * TS::NHALO, src + v * a.ndof);
  }
  if (in[D] == N - 1 && lc[D] == teff[D] - 1) {
    const double* src = a.Win + (g + off1);
#pragma unroll
    for (int v = 0; v < 5; ++v) dg_async_copy8(dst + FPD + v * TS::NHALO, src + v * a.ndof);
  }
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

// HLL flux (reading R9, Eq. 21-24) at face point fl of direction D from the node records of its two
// sides:  F = cL F_L + cR F_R + cU (U_R - U_L),  F_s = U_s v_s + P_s e_D (+ P_s v_s in the energy).
template <int ND, int N, int D>
__device__ __forceinline__ void dg_face_flux(const double* X, const double* XH, double* Fh, int fl,
                                             const int teff[3]) {
  using TS = TileShape<ND, N>;
  using DI = DirInfo<ND, N, D>;
  constexpr int A = DI::A, B = DI::B, FPD = DI::FPD, ST = TS::NTN, SH = TS::NHALO;
  const int p = fl / FPD, fp = fl - p * FPD;
  int la, lb, ca, cb;
  DI::split(fp, la, lb, ca, cb);
  if (p > teff[D] || la >= teff[A] || lb >= teff[B]) return;
  const int tnode = ca * TS::SN(A) + cb * TS::SN(B);
  const int telem = la * TS::SE(A) + lb * TS::SE(B);
  // left / right records: a tile node (stride ST, rows v=5+D P=8 num=9 den=10) or a halo point
  // (stride SH, rows v=5 P=6 num=7 den=8)
  const bool hL = (p < 1), hR = (p >= teff[D]);
  const double* xl = hL ? XH + (TS::HOFF(D) + fp)
                        : X + ((telem + (p - 1) * TS::SE(D)) * TS::NN + tnode + (N - 1) * TS::SN(D));
  const double* xr = hR ? XH + (TS::HOFF(D) + FPD + fp) : X + ((telem + p * TS::SE(D)) * TS::NN + tnode);
  const int sl = hL ? SH : ST, sr = hR ? SH : ST;
  const double* ql = xl + (hL ? 5 * SH : (5 + D) * ST);              // v, then (P, num, den) at +kl
  const double* qr = xr + (hR ? 5 * SH : (5 + D) * ST);
  const int kl = hL ? SH : (3 - D) * ST, kr = hR ? SH : (3 - D) * ST;
  const double vL = ql[0], vR = qr[0];
  const double PL = ql[kl], PR = qr[kr];
  double nmL, npL, dL, nmR, npR, dR;
  {
    const double num = ql[kl + sl], den = ql[kl + 2 * sl];
    const double root = dg_sqrt(num * fma(fma(-vL, vL, 1.0), den, num));
    const double c = vL * den;
    nmL = c - root; npL = c + root; dL = den + num;
  }
  {
    const double num = qr[kr + sr], den = qr[kr + 2 * sr];
    const double root = dg_sqrt(num * fma(fma(-vR, vR, 1.0), den, num));
    const double c = vR * den;
    nmR = c - root; npR = c + root; dR = den + num;
  }
  const bool ml = nmL * dR <= nmR * dL, mr = npL * dR >= npR * dL;       // Eq. 23-24 by cross-multiplication
  const double nl = ml ? nmL : nmR, dl = ml ? dL : dR;
  const double nr = mr ? npL : npR, dr = mr ? dL : dR;
  double cL, cR, cU;
  if (nl >= 0.0) { cL = 1.0; cR = 0.0; cU = 0.0; }
  else if (nr <= 0.0) { cL = 0.0; cR = 1.0; cU = 0.0; }
  else {
    const double aa = nr * dl, bb = nl * dr;
    const double q = dg_rcp(aa - bb);
    cL = aa * q; cR = -bb * q; cU = nl * nr * q;
  }
  const double kL = fma(cL, vL, -cU), kR = fma(cR, vR, cU);
  const double pL = cL * PL, pR = cR * PR;
  double* pF = Fh + 5 * TS::FOFF(D) + p * 5 * FPD + fp;
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    double f = fma(kL, xl[v * sl], kR * xr[v * sr]);
    if (v == 1 + D) f += pL + pR;
    if (v == 4) f = fma(pL, vL, fma(pR, vR, f));
    pF[v * FPD] = f;
  }
}

// Volume term of direction D for this thread's node (Eq. 17 over the diagonal mass matrix): the
// tensor-line contraction of F_D(W_q) = U_q v_q + P_q e_D, formed on the fly from the node records.
template <int ND, int N, int D>
__device__ __forceinline__ void dg_volume(const StageArgs& a, const double* sD, const double* X, int ti,
                                          const int in[3], double R[5]) {
  using TS = TileShape<ND, N>;
  constexpr int NTOT = TS::NTN;
  const int id = in[D];
  const double* line = X + (ti - id * TS::SN(D));
  const double* dh = sD + id * N;
#pragma unroll
  for (int q = 0; q < N; ++q) {
    const double* x = line + q * TS::SN(D);
    const double dq = a.rh[D] * dh[q];
    const double t = dq * x[(5 + D) * NTOT];
    const double Pq = x[8 * NTOT];
#pragma unroll
    for (int v = 0; v < 5; ++v) R[v] = fma(t, x[v * NTOT], R[v]);
    R[1 + D] = fma(dq, Pq, R[1 + D]);
    R[4] = fma(t, Pq, R[4]);
  }
}


// Physicality operator on the cells of one warp group (PAPER.md:242-252 steps 1-4); a thread owns the
// M nodes n0 + m NNT of its cell (tile slots ti0 + m NNT).  Cell-local reductions go through shared
// memory with group barriers only.  Must be called by every thread of the group.  Uo: the nodes'
// states, limited in place.
template <int ND, int N>
__device__ __forceinline__ void dg_limiter_group(double (*Uo)[5], bool active, int ti0, int le, int n0,
                                                 int grp, const double* wn, const StageArgs& a,
                                                 double* scratch, double* sPart, double* sMean,
                                                 dg_ull* sSmin, int* sFlag, int* sCnt) {
  using TS = TileShape<ND, N>;
  constexpr int NN = TS::NN, NTN = TS::NTN, M = TS::M, NNT = TS::NNT;
  bool bad = false;
  if (active) {
#pragma unroll
    for (int m = 0; m < M; ++m) bad = bad || !dg_admissible(Uo[m], a.f_screen);   // step 1: screen (R13e)
  }
  if (bad) sFlag[le] = 1;
  dg_gsync<TS::G>(grp);
  const bool flagged = active && (sFlag[le] != 0);
  // nothing flagged in this warp group (the common case): done, no further group barriers
  const bool any = (TS::G == 1) ? (__any_sync(0xffffffffu, flagged) != 0) : (sFlag[grp * TS::EPG] != 0);
  if (!any) return;
  if (flagged) {
#pragma unroll
    for (int m = 0; m < M; ++m) {
#pragma unroll
      for (int v = 0; v < 5; ++v) scratch[v * NTN + ti0 + m * NNT] = wn[m] * Uo[m][v];
    }
  }
  dg_gsync<TS::G>(grp);
  // cell average: J interleaved partial sums per variable (5 J lanes), then their sum by 5 lanes
  constexpr int J = (NNT >= 20) ? 4 : NNT / 5;
  if (J == 0) {                                                     // tiny cells: one lane sums
    if (flagged && n0 == 0) {
      for (int v = 0; v < 5; ++v) {
        double acc = 0.0;
        for (int q = 0; q < NN; ++q) acc += scratch[v * NTN + le * NN + q];
        sMean[le * 5 + v] = acc / a.wsum;
      }
    }
  } else {
    if (flagged && n0 < 5 * J) {
      const int v = n0 % 5, j = n0 / 5;
      const double* p = scratch + v * NTN + le * NN;
      double acc = 0.0;
      for (int q = j; q < NN; q += J) acc += p[q];
      sPart[le * 20 + n0] = acc;
    }
    dg_gsync<TS::G>(grp);
    if (flagged && n0 < 5) {
      double acc = 0.0;
#pragma unroll
      for (int j = 0; j < J; ++j) acc += sPart[le * 20 + 5 * j + n0];
      sMean[le * 5 + n0] = acc / a.wsum;
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
      si = 1.0;
#pragma unroll
      for (int m = 0; m < M; ++m) {
        double sm_ = dg_limiter_node_s(Ub, Uo[m], a.f_solve);        // step 3
        if (!(sm_ >= 0.0)) sm_ = 0.0;
        si = fmin(si, sm_);
      }
    }
    if (si < 1.0) atomicMin(&sSmin[le], dg_ord(si));                 // step 4: s = min_i s_i
    if (n0 == 0) {
      atomicAdd(&sCnt[0], 1);
      if (!mean_ok) atomicAdd(&sCnt[1], 1);
    }
  }
  dg_gsync<TS::G>(grp);
  if (flagged) {
    const double s = a.one_m_delta * dg_unord(sSmin[le]);            // R13c
    const double tt = 1.0 - s;
#pragma unroll
    for (int m = 0; m < M; ++m) {
#pragma unroll
      for (int v = 0; v < 5; ++v)                                    // Eq. 26 from the nearer end (R14)
        Uo[m][v] = (s > 0.5) ? fma(tt, Ub[v] - Uo[m][v], Uo[m][v]) : fma(s, Uo[m][v] - Ub[v], Ub[v]);
    }
  }
}

// resident blocks per SM the register allocation must allow: up to 1024 threads (32 warps) per SM,
// but no more blocks than the shared memory of an SM holds
#ifndef DG_MINB
#define DG_MINB TileShape<ND, N>::MINB
#endif
template <int ND, int N, int EOS>
__global__ void __launch_bounds__(TileShape<ND, N>::NT, DG_MINB)
dg_stage_kernel(const __grid_constant__ StageArgs a) {
  using TS = TileShape<ND, N>;
  constexpr int NN = TS::NN, NTN = TS::NTN, NT = TS::NT, NE = TS::NE;
  extern __shared__ __align__(16) double sm[];
  double* X = sm + TS::O_X;
  double* XH = sm + TS::O_XH;
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
  // warp group, element and the M nodes (n0 + m NNT) of this thread
  constexpr int M = TS::M, NNT = TS::NNT;
  const int t = threadIdx.x;
  const int grp = t / TS::GT, r = t - grp * TS::GT;
  const int le = grp * TS::EPG + r / NNT, n0 = r % NNT;
  const int ti0 = le * NN + n0;                                      // tile slot of node m: ti0 + m NNT
  const int lc[3] = {le % TS::TX, (le / TS::TX) % TS::TY, le / (TS::TX * TS::TY)};
  const bool active = (r < TS::EPG * NNT) && lc[0] < teff[0] && lc[1] < teff[1] && lc[2] < teff[2];
  int g0 = 0;                                                        // ndof < 2^31 (dgrhd_create)
  if (active) g0 = ((org[0] + lc[0]) + a.ne[0] * ((org[1] + lc[1]) + a.ne[1] * (org[2] + lc[2]))) * NN + n0;
  int in[M][3];
#pragma unroll
  for (int m = 0; m < M; ++m) {
    const int n = n0 + m * NNT;
    in[m][0] = n % N; in[m][1] = (n / N) % N; in[m][2] = n / (N * N);
  }
  if (t < NE) { sSmin[t] = dg_ord(1.0); sFlag[t] = 0; }
  if (t < 4) sCnt[t] = 0;
  if (t < N * N) sD[t] = a.Dhat[t];

  // 1. primitives (recovered by the previous stage) and conserved state of the nodes -> their records
  //    in the shared node array; primitives of the neighbours' facing nodal layers -> halo slots
#pragma unroll
  for (int m = 0; m < M; ++m) {
    dg_load_halo<ND, N, 0>(a, XH, active, g0 + m * NNT, lc, in[m], org, teff);
    if constexpr (ND > 1) dg_load_halo<ND, N, 1>(a, XH, active, g0 + m * NNT, lc, in[m], org, teff);
    if constexpr (ND > 2) dg_load_halo<ND, N, 2>(a, XH, active, g0 + m * NNT, lc, in[m], org, teff);
  }
  double Un[M][5];
#pragma unroll
  for (int m = 0; m < M; ++m)
#pragma unroll
    for (int v = 0; v < 5; ++v) Un[m][v] = 0.0;
  if (active) {
    double Wn[M][5];
#pragma unroll
    for (int m = 0; m < M; ++m) {
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        Wn[m][v] = __ldg(a.Win + v * a.ndof + g0 + m * NNT);
        Un[m][v] = a.Us[v * a.ndof + g0 + m * NNT];
      }
    }
#pragma unroll
    for (int m = 0; m < M; ++m) dg_node_record<ND, N, EOS>(a.eos, Wn[m], Un[m], X, ti0 + m * NNT);
    if (a.mode == DG_MODE_STAGE && a.a != 0.0) {         // U0 is needed last: warm L2 now
#pragma unroll
      for (int m = 0; m < M; ++m)
#pragma unroll
        for (int v = 0; v < 5; ++v)
          asm volatile("prefetch.global.L2 [%0];" ::"l"(a.U0 + v * a.ndof + g0 + m * NNT));
    }
  }
  dg_async_wait();
  __syncthreads();
  // records of the halo points (U from W by Eq. 4, reading R8), a dense pass over the halo slots
  for (int h = t; h < TS::NHALO; h += NT) dg_halo_record<ND, N, EOS>(a.eos, XH, h);
  __syncthreads();

  // 2. interface flux at every face point of the tile, once each, spread over all threads
  for (int f = t; f < TS::NFACE; f += NT) {
    if (ND == 1 || f < TS::FOFF(1)) dg_face_flux<ND, N, 0>(X, XH, Fh, f, teff);
    else if (ND == 2 || f < TS::FOFF(2)) dg_face_flux<ND, N, (ND > 1 ? 1 : 0)>(X, XH, Fh, f - TS::FOFF(1), teff);
    else dg_face_flux<ND, N, (ND > 2 ? 2 : 0)>(X, XH, Fh, f - TS::FOFF(2), teff);
  }

  // 3. volume quadrature: reads the node array only, so it needs no barrier and fills the time
  //    other warps still spend on face fluxes
  double R[M][5];
#pragma unroll
  for (int m = 0; m < M; ++m)
#pragma unroll
    for (int v = 0; v < 5; ++v) R[m][v] = 0.0;
  if (active) {
#pragma unroll
    for (int m = 0; m < M; ++m) {
      dg_volume<ND, N, 0>(a, sD, X, ti0 + m * NNT, in[m], R[m]);
      if constexpr (ND > 1) dg_volume<ND, N, 1>(a, sD, X, ti0 + m * NNT, in[m], R[m]);
      if constexpr (ND > 2) dg_volume<ND, N, 2>(a, sD, X, ti0 + m * NNT, in[m], R[m]);
    }
  }
  __syncthreads();

  // 4. surface lift
  if (active) {
#pragma unroll
    for (int m = 0; m < M; ++m) {
      dg_add_surface<ND, N, 0>(Fh, lc, in[m], a.rh[0] * a.lift, R[m]);
      if constexpr (ND > 1) dg_add_surface<ND, N, 1>(Fh, lc, in[m], a.rh[1] * a.lift, R[m]);
      if constexpr (ND > 2) dg_add_surface<ND, N, 2>(Fh, lc, in[m], a.rh[2] * a.lift, R[m]);
    }
  }
  if (a.mode == DG_MODE_RHS) {
    if (active) {
#pragma unroll
      for (int m = 0; m < M; ++m)
#pragma unroll
        for (int v = 0; v < 5; ++v) a.Rout[v * a.ndof + g0 + m * NNT] = R[m][v];
    }
    return;
  }

  // 5. SSP-RK combine (Shu-Osher form)
  const double dt = *a.dt_ptr;
  double Uo[M][5];
#pragma unroll
  for (int m = 0; m < M; ++m)
#pragma unroll
    for (int v = 0; v < 5; ++v) Uo[m][v] = a.b * fma(dt, R[m][v], Un[m][v]);
  if (a.a != 0.0 && active) {
#pragma unroll
    for (int m = 0; m < M; ++m)
#pragma unroll
      for (int v = 0; v < 5; ++v) Uo[m][v] = fma(a.a, a.U0[v * a.ndof + g0 + m * NNT], Uo[m][v]);
  }

  // 6. physicality-enforcing operator (cell-local; the node array is free after the barrier above)
  double wn[M];
#pragma unroll
  for (int m = 0; m < M; ++m) {
    wn[m] = a.w[in[m][0]];
    if (ND > 1) wn[m] *= a.w[in[m][1]];
    if (ND > 2) wn[m] *= a.w[in[m][2]];
  }
  dg_limiter_group<ND, N>(Uo, active, ti0, le, n0, grp, wn, a, X, sPart, sMean, sSmin, sFlag, sCnt);

  // 7. primitives of the new state, CFL maximum
  double speed = 0.0;
  if (active) {
    double Wo[M][5];
#pragma unroll
    for (int m = 0; m < M; ++m) {
      const int st = dg_con2prim<EOS>(a.eos, Uo[m], Wo[m]);
      if (st != 0) atomicAdd(&sCnt[2], 1);
    }
#pragma unroll
    for (int m = 0; m < M; ++m)
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        a.Uout[v * a.ndof + g0 + m * NNT] = Uo[m][v];
        a.Wout[v * a.ndof + g0 + m * NNT] = Wo[m][v];
      }
    if (a.do_cfl) {
#pragma unroll
      for (int m = 0; m < M; ++m) {
        const double sp = dg_cfl_speed<EOS, ND>(a.eos, Wo[m], a.cw);
        if (sp > 0.0) speed = fmax(speed, sp);
      }
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

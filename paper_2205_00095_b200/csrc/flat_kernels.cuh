// flat_kernels.cuh -- the point-wise and cell-wise kernels of the CUDA path that need no
// neighbour data (sm_100a, fp64):
//   dg_c2p_batch_kernel    conserved -> primitive over a flat SoA batch
//   dg_p2c_batch_kernel    primitive -> conserved (Eq. 4)
//   dg_c2p_state_kernel    pressure (and optionally all primitives) of a context state, the failure
//                          counter and the CFL wave-speed maximum (reading R11)
//   dg_limiter_kernel      the physicality-enforcing operator on caller data:
//                          the SAME device function as inside the fused stage kernel
//   dg_dt_kernel           dt = cfl / amax on the device (no host round trip)
// All are HBM-streaming kernels.  The batch kernels give each thread NS = 2 adjacent states: one
// 16-byte access per variable and thread (a warp moves 512 contiguous bytes per row) and two
// independent solver streams.
#pragma once
#include "stage_kernel.cuh"

#define DG_FLAT_NT 256

// fallbacks of the Taub-Matthews solve (physics.cuh) taken by the context-free batch calls
__device__ dg_ull g_tm_fallbacks;

// block-wide max of a non-negative double -> one atomicMax on its ordered-integer image
__device__ __forceinline__ void dg_block_atomic_max(double x, double* sRed, dg_ull* dst) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x = fmax(x, __shfl_xor_sync(0xffffffffu, x, o));
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) sRed[wid] = x;
  __syncthreads();
  if (wid == 0) {
    const int nw = (blockDim.x + 31) >> 5;
    double y = (lane < nw) ? sRed[lane] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) y = fmax(y, __shfl_xor_sync(0xffffffffu, y, o));
    if (lane == 0 && y > 0.0) atomicMax(dst, dg_ord(y));
  }
}

// NS = 2: n even and U, W 16-byte aligned (checked by the host); NS = 1: any n / alignment.
// Resident blocks per SM (measured at 2^26 states): the ideal-EOS solve wants 80 registers (no spills, 3 blocks:
// 0.86 of HBM against 0.82 with 4 blocks and 64 registers), the Taub-Matthews solve fits 64 (4 blocks: 0.86).
template <int EOS, int NS>
__global__ void __launch_bounds__(DG_FLAT_NT, (EOS == DG_EOS_IDEAL) ? 3 : 4)
dg_c2p_batch_kernel(long long n, const double* __restrict__ U, double* __restrict__ W,
                    int* __restrict__ status, EosPar eos) {
  const long long i = ((long long)blockIdx.x * DG_FLAT_NT + threadIdx.x) * NS;
  if (i >= n) return;
  double u[NS][5], w[NS][5];
  int st[NS], nfall = 0;
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    double x[NS];
    dg_ldg_line<NS>(U + v * n + i, x);
#pragma unroll
    for (int s = 0; s < NS; ++s) u[s][v] = x[s];
  }
  dg_con2prim_n<EOS, NS, true>(eos, u, w, nullptr, st, &nfall);
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    double x[NS];
#pragma unroll
    for (int s = 0; s < NS; ++s) x[s] = w[s][v];
    dg_st_line<NS>(W + v * n + i, x);
  }
  if (status) {
#pragma unroll
    for (int s = 0; s < NS; ++s) status[i + s] = st[s];
  }
  if (EOS == DG_EOS_TM && nfall) atomicAdd(&g_tm_fallbacks, (dg_ull)nfall);
}

// (the comparison variants of con2prim live in c2p_variant.cu, compiled without FMA contraction)

template <int EOS>
__global__ void __launch_bounds__(DG_FLAT_NT)
dg_p2c_batch_kernel(long long n, const double* __restrict__ W, double* __restrict__ U, EosPar eos) {
  const long long i = (long long)blockIdx.x * DG_FLAT_NT + threadIdx.x;
  if (i >= n) return;
  double u[5], w[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) w[v] = __ldg(W + v * n + i);
  dg_prim2con<EOS>(eos, w, u);
#pragma unroll
  for (int v = 0; v < 5; ++v) U[v * n + i] = u[v];
}

// P = P(U) at every node of a state (Eq. 16), P / W optional outputs (W: all five primitives).
// counters (or NULL): [2] += failures, [3] += Taub-Matthews fallbacks.  amax (or NULL): atomicMax of
// sum_d cw[d] max(|lambda-_d|,|lambda+_d|) over the nodes (R11).
template <int EOS, int ND>
__global__ void __launch_bounds__(DG_FLAT_NT)
dg_c2p_state_kernel(long long n, const double* __restrict__ U, double* __restrict__ P,
                    double* __restrict__ W, EosPar eos, double cw0, double cw1, double cw2,
                    dg_ull* amax, dg_ull* counters) {
  __shared__ double sRed[32];
  __shared__ int sFail[2];
  if (threadIdx.x < 2) sFail[threadIdx.x] = 0;
  __syncthreads();
  const long long i = (long long)blockIdx.x * DG_FLAT_NT + threadIdx.x;
  double speed = 0.0;
  if (i < n) {
    double u[1][5], w[1][5];
    int st[1], nfall = 0;
#pragma unroll
    for (int v = 0; v < 5; ++v) u[0][v] = __ldg(U + v * n + i);
    dg_con2prim_n<EOS, 1, true>(eos, u, w, nullptr, st, &nfall);
    if (P) P[i] = w[0][4];
    if (W) {
#pragma unroll
      for (int v = 0; v < 5; ++v) W[v * n + i] = w[0][v];
    }
    if (st[0] != 0) atomicAdd(&sFail[0], 1);
    if (nfall) atomicAdd(&sFail[1], nfall);
    if (amax) {
      const double cw[3] = {cw0, cw1, cw2};
      const double s = dg_cfl_speed<EOS, ND>(eos, u[0], w[0][4], cw);
      if (s > 0.0) speed = s;                       // NaN never wins
    }
  }
  if (amax) dg_block_atomic_max(speed, sRed, amax + (blockIdx.x % DG_NSLOT) * DG_SLOT_STRIDE);
  __syncthreads();
  if (threadIdx.x == 0 && counters) {
    const int slot = (blockIdx.x % DG_NSLOT) * DG_SLOT_STRIDE;
    if (sFail[0]) atomicAdd(&counters[slot + 2], (dg_ull)sFail[0]);
    if (sFail[1]) atomicAdd(&counters[slot + 3], (dg_ull)sFail[1]);
  }
}

// The physicality-enforcing operator on a canonical-layout state: the thread mapping of the fused
// stage kernel (a thread owns a segment of an x-line, a cell is NL consecutive lanes of one warp) over
// a flat list of cells.  flag[n_e] / s[n_e] optional; counters[0..1] += flagged cells / inadmissible
// means.
template <int ND, int N>
__global__ void __launch_bounds__(128)
dg_limiter_kernel(long long nelem, long long ndof, double* U, unsigned char* flag, double* s_out,
                  LimPar lp, dg_ull* counters) {
  using TS = TileShape<ND, N>;
  constexpr int NN = TS::NN, NL = TS::NL, EPW = TS::EPW, SEG = TS::SEG, NSEG = TS::NSEG;
  const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
  const int ew = lane / NL, lt = lane - ew * NL;
  const int h = lt % NSEG, ln = lt / NSEG;
  const long long e = ((long long)blockIdx.x * 4 + wrp) * EPW + ew;
  const bool active = (ew < EPW) && (e < nelem);
  const int j = (ND >= 2) ? ln % N : 0, k = (ND >= 3) ? ln / N : 0;
  const long long g0 = e * NN + N * ln + h * SEG;
  double Uo[SEG][5];
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    double x[SEG];
    if (active) dg_ld_line<SEG>(U + v * ndof + g0, x);
#pragma unroll
    for (int m = 0; m < SEG; ++m) Uo[m][v] = active ? x[m] : 0.0;
  }
  double wl = 1.0;
  if (ND >= 2) wl *= lp.w[j];
  if (ND >= 3) wl *= lp.w[k];
  double wn[SEG];
#pragma unroll
  for (int m = 0; m < SEG; ++m) wn[m] = wl * ((NSEG > 1 && h > 0) ? lp.w[(SEG + m) % 5] : lp.w[m]);
  int cnt[2] = {0, 0};
  double s;
  const bool flagged = dg_limiter_cells<NL, SEG>(Uo, active, lane, wn, lp, cnt, s);
  if (active && flagged) {
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      double x[SEG];
#pragma unroll
      for (int m = 0; m < SEG; ++m) x[m] = Uo[m][v];
      dg_st_line<SEG>(U + v * ndof + g0, x);
    }
  }
  if (active && lt == 0) {
    if (flag) flag[e] = flagged ? 1 : 0;
    if (s_out) s_out[e] = s;
  }
  if (counters) {
    if (cnt[0]) atomicAdd(&counters[0], (dg_ull)cnt[0]);
    if (cnt[1]) atomicAdd(&counters[1], (dg_ull)cnt[1]);
  }
}

// ---------------------------------------------------------------------------------------------
// Shock limiter of Moe, Rossmanith & Seal (PAPER.md:126, :551, :621 ref [23]; reading R18:
// cited, not printed, by the paper).  Two cell-wise kernels in the thread mapping of the stage kernel
// (a cell = NL consecutive lanes of one warp, reductions by shuffle), run after a stage when the
// context's shock_limiter is on:
//   dg_moe_stats_kernel   per cell and conserved variable: average (tensor GLL weights), maximum and
//                         minimum over the cell's nodes            -> stats[n_e][15]
//   dg_moe_apply_kernel   bounds from the face neighbours' extrema (periodic wrap; none beyond any
//                         other boundary) and the tolerance alpha; theta = min(1, phi(.)) over all
//                         variables, phi(y) = min(y/1.1, 1); U <- Ubar + theta (U - Ubar) in the limited
//                         cells, whose pressure is recovered again; on the step's last stage the CFL
//                         maximum is taken here, from the limited state.  LIMK = 1: theta of the
//                         minmod limiter (dg_mm_theta, statistics of dg_mm_stats_kernel) instead.
// ---------------------------------------------------------------------------------------------
template <int NL>
DG_INL double dg_cell_max(double x, int base) {
  if ((NL & (NL - 1)) == 0) {
#pragma unroll
    for (int o = NL / 2; o > 0; o >>= 1) x = fmax(x, __shfl_xor_sync(0xffffffffu, x, o));
    return x;
  }
  double acc = x;
#pragma unroll
  for (int o = 0; o < NL; ++o) acc = fmax(acc, __shfl_sync(0xffffffffu, x, min(base + o, 31)));
  return acc;
}

template <int ND, int N>
__global__ void __launch_bounds__(128)
dg_moe_stats_kernel(long long nelem, long long ndof, const double* __restrict__ U, double* __restrict__ stats,
                    LimPar lp) {
  using TS = TileShape<ND, N>;
  constexpr int NN = TS::NN, NL = TS::NL, EPW = TS::EPW, SEG = TS::SEG, NSEG = TS::NSEG;
  const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
  const int ew = lane / NL, lt = lane - ew * NL;
  const int h = lt % NSEG, ln = lt / NSEG;
  const long long e = ((long long)blockIdx.x * 4 + wrp) * EPW + ew;
  const bool active = (ew < EPW) && (e < nelem);
  const int j = (ND >= 2) ? ln % N : 0, k = (ND >= 3) ? ln / N : 0;
  const long long g0 = (active ? e : 0) * NN + N * ln + h * SEG;
  const int base = ew * NL;
  double wl = 1.0;
  if (ND >= 2) wl *= lp.w[j];
  if (ND >= 3) wl *= lp.w[k];
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    double x[SEG];
    dg_ld_line<SEG>(U + v * ndof + g0, x);
    double part = 0.0, mx = x[0], mn = x[0];
#pragma unroll
    for (int m = 0; m < SEG; ++m) {
      const double wq = wl * ((NSEG > 1 && h > 0) ? lp.w[(SEG + m) % 5] : lp.w[m]);
      part = fma(wq, x[m], part);
      mx = fmax(mx, x[m]);
      mn = fmin(mn, x[m]);
    }
    const double mean = dg_cell_sum<NL>(part, base) / lp.wsum;
    mx = dg_cell_max<NL>(mx, base);
    mn = dg_cell_min<NL>(mn, base);
    if (active && lt == 0) {
      stats[e * 15 + v] = mean;
      stats[e * 15 + 5 + v] = mx;
      stats[e * 15 + 10 + v] = mn;
    }
  }
}

// Minmod limiter (PAPER.md:126, :597 ref [24]; reading R19: cited, not printed): statistics per
// cell and conserved variable -> stats[n_e][25] = average[5] | linear coefficients a_d[3][5] | max|w|[5],
//   a_d = sum_n w_n xi_d(n) w(n) / sum_n w_n xi_d(n)^2   (tensor GLL weights; rxx = 1 / that denominator).
struct MmPar {
  double x[5];      // GLL nodes on [-1,1]
  double rxx;
};

template <int ND, int N>
__global__ void __launch_bounds__(128)
dg_mm_stats_kernel(long long nelem, long long ndof, const double* __restrict__ U, double* __restrict__ stats,
                   LimPar lp, MmPar mm) {
  using TS = TileShape<ND, N>;
  constexpr int NN = TS::NN, NL = TS::NL, EPW = TS::EPW, SEG = TS::SEG, NSEG = TS::NSEG;
  const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
  const int ew = lane / NL, lt = lane - ew * NL;
  const int h = lt % NSEG, ln = lt / NSEG;
  const long long e = ((long long)blockIdx.x * 4 + wrp) * EPW + ew;
  const bool active = (ew < EPW) && (e < nelem);
  const int j = (ND >= 2) ? ln % N : 0, k = (ND >= 3) ? ln / N : 0;
  const long long g0 = (active ? e : 0) * NN + N * ln + h * SEG;
  const int base = ew * NL;
  double wl = 1.0;
  if (ND >= 2) wl *= lp.w[j];
  if (ND >= 3) wl *= lp.w[k];
  const double xy = (ND >= 2) ? mm.x[j] : 0.0, xz = (ND >= 3) ? mm.x[k] : 0.0;
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    double x[SEG];
    dg_ld_line<SEG>(U + v * ndof + g0, x);
    double pm = 0.0, px = 0.0, big = 0.0;
#pragma unroll
    for (int m = 0; m < SEG; ++m) {
      const int i = (NSEG > 1 && h > 0) ? (SEG + m) % 5 : m;
      const double wq = wl * lp.w[i];
      pm = fma(wq, x[m], pm);
      px = fma(wq * mm.x[i], x[m], px);
      big = fmax(big, fabs(x[m]));
    }
    const double mean = dg_cell_sum<NL>(pm, base) / lp.wsum;
    const double ax = dg_cell_sum<NL>(px, base) * mm.rxx;
    const double ay = (ND >= 2) ? dg_cell_sum<NL>(pm * xy, base) * mm.rxx : 0.0;
    const double az = (ND >= 3) ? dg_cell_sum<NL>(pm * xz, base) * mm.rxx : 0.0;
    big = dg_cell_max<NL>(big, base);
    if (active && lt == 0) {
      stats[e * 25 + v] = mean;
      stats[e * 25 + 5 + v] = (N > 1) ? ax : 0.0;
      stats[e * 25 + 10 + v] = (N > 1) ? ay : 0.0;
      stats[e * 25 + 15 + v] = (N > 1) ? az : 0.0;
      stats[e * 25 + 20 + v] = big;
    }
  }
}

// Neighbour of cell e along axis d on side `side` (0 minus, 1 plus): its index, or -1 when there is none
// (periodic wrap; no neighbour beyond any other boundary).  Cell indices fit 32 bits (ndof < 2^31).
DG_INL int dg_cell_neighbour(int e, const int ie[3], const int ne[3], const int periodic[3], int d, int side) {
  const int es = (d == 0) ? 1 : (d == 1 ? ne[0] : ne[0] * ne[1]);
  int jd = ie[d] + (side ? 1 : -1);
  if (jd < 0 || jd >= ne[d]) {
    if (!periodic[d]) return -1;
    jd = (jd < 0) ? ne[d] - 1 : 0;
  }
  return e + (jd - ie[d]) * es;
}

// theta of the minmod limiter (reading R19) from ONE variable v of cell e: min over the directions of
// minmod(a_d, beta D+/2, beta D-/2) / a_d, D+- the differences of the neighbouring cell averages (a missing
// neighbour drops out).  The cell's theta is the minimum over v, set to 1 if >= 1 - 1e-12 (by the caller).
template <int ND>
DG_INL double dg_mm_theta_var(const double* __restrict__ stats, int e, int v, const int ie[3], const int ne[3],
                              const int periodic[3], double beta) {
  const double wb = stats[(long long)e * 25 + v], tiny = 1e-12 * stats[(long long)e * 25 + 20 + v];
  double theta = 1.0;
#pragma unroll
  for (int d = 0; d < ND; ++d) {
    const double a = stats[(long long)e * 25 + 5 + 5 * d + v];
    if (!(fabs(a) > tiny)) continue;
    const double sg = (a > 0.0) ? 1.0 : -1.0;
    double m = fabs(a);
    bool zero = false;
#pragma unroll
    for (int side = 0; side < 2; ++side) {
      const int en = dg_cell_neighbour(e, ie, ne, periodic, d, side);
      if (en < 0) continue;
      const double wn = stats[(long long)en * 25 + v];
      const double b = 0.5 * beta * (side ? wn - wb : wb - wn);
      if (b * sg <= 0.0) zero = true;
      m = fmin(m, fabs(b));
    }
    const double r = zero ? 0.0 : (sg * m) / a;
    theta = fmin(theta, r);
  }
  return theta;
}

// theta of the Moe limiter (reading R18) from ONE variable v of cell e: bounds from the face neighbours'
// extrema and the tolerance alpha, phi(y) = min(y/1.1, 1) on both sides.
template <int ND>
DG_INL double dg_moe_theta_var(const double* __restrict__ stats, int e, int v, const int ie[3], const int ne[3],
                               const int periodic[3], double alpha) {
  const double wb = stats[(long long)e * 15 + v], wM = stats[(long long)e * 15 + 5 + v], wm = stats[(long long)e * 15 + 10 + v];
  double M = wb + alpha, m = wb - alpha;
#pragma unroll
  for (int d = 0; d < ND; ++d)
#pragma unroll
    for (int side = 0; side < 2; ++side) {
      const int en = dg_cell_neighbour(e, ie, ne, periodic, d, side);
      if (en < 0) continue;
      M = fmax(M, stats[(long long)en * 15 + 5 + v]);
      m = fmin(m, stats[(long long)en * 15 + 10 + v]);
    }
  const double tiny = 1e-12 * fmax(fabs(wM), fabs(wm));     // extremum = mean to rounding: no limit
  const double tM = (wM - wb > tiny) ? fmin((M - wb) / (wM - wb) / 1.1, 1.0) : 1.0;
  const double tm = (wb - wm > tiny) ? fmin((wb - m) / (wb - wm) / 1.1, 1.0) : 1.0;
  return fmin(tM, tm);
}

struct MoePar {
  long long ne[3];
  int periodic[3];
  double alpha;          // Moe: tolerance alpha; minmod: beta
  double cw[3];
  int do_cfl;
};

template <int ND, int N, int EOS, int LIMK>
__global__ void __launch_bounds__(128)
dg_moe_apply_kernel(long long nelem, long long ndof, double* U, double* P, const double* __restrict__ stats,
                    MoePar mp, EosPar eos, dg_ull* amax, dg_ull* counters, double* theta_out) {
  using TS = TileShape<ND, N>;
  constexpr int NN = TS::NN, NL = TS::NL, EPW = TS::EPW, SEG = TS::SEG, NSEG = TS::NSEG;
  const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
  const int ew = lane / NL, lt = lane - ew * NL;
  const int h = lt % NSEG, ln = lt / NSEG;
  const long long e = ((long long)blockIdx.x * 4 + wrp) * EPW + ew;
  const bool active = (ew < EPW) && (e < nelem);
  const long long g0 = (active ? e : 0) * NN + N * ln + h * SEG;
  // theta: lane v of the cell takes variable v (its own and its face neighbours' statistics), the cell's
  // lanes then share the minimum.  (Every lane working through all five variables, with 64-bit index
  // arithmetic, made this kernel cost as much as a stage: 6.7 ms at 128^3, p = 3.)
  double th = 1.0;
  if (active && lt < 5) {
    const int ei = (int)e, ne[3] = {(int)mp.ne[0], (int)mp.ne[1], (int)mp.ne[2]};
    const int ie[3] = {ei % ne[0], (ei / ne[0]) % ne[1], ei / (ne[0] * ne[1])};
    for (int v = lt; v < 5; v += NL)
      th = fmin(th, LIMK == 1 ? dg_mm_theta_var<ND>(stats, ei, v, ie, ne, mp.periodic, mp.alpha)
                              : dg_moe_theta_var<ND>(stats, ei, v, ie, ne, mp.periodic, mp.alpha));
  }
  double theta = dg_cell_min<NL>(th, ew * NL);
  if (LIMK == 1) theta = (theta >= 1.0 - 1e-12) ? 1.0 : theta;
  double mean[5] = {0, 0, 0, 0, 0};
  if (active && theta < 1.0) {
#pragma unroll
    for (int v = 0; v < 5; ++v) mean[v] = stats[e * (LIMK == 1 ? 25 : 15) + v];
  }
  if (theta_out && active && lt == 0) theta_out[e] = theta;
  const bool lim = active && (theta < 1.0);
  const bool need = lim || (active && mp.do_cfl);
  double speed = 0.0;
  int nfail = 0, nfall = 0;
  if (need) {
    double Uo[SEG][5], Po[SEG];
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      double x[SEG];
      dg_ld_line<SEG>(U + v * ndof + g0, x);
#pragma unroll
      for (int m = 0; m < SEG; ++m) Uo[m][v] = lim ? fma(theta, x[m] - mean[v], mean[v]) : x[m];
    }
    if (lim) {
      int st[SEG];
      dg_con2prim_n<EOS, SEG, false>(eos, Uo, nullptr, Po, st, &nfall);
#pragma unroll
      for (int m = 0; m < SEG; ++m) nfail += (st[m] != 0) ? 1 : 0;
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        double x[SEG];
#pragma unroll
        for (int m = 0; m < SEG; ++m) x[m] = Uo[m][v];
        dg_st_line<SEG>(U + v * ndof + g0, x);
      }
      dg_st_line<SEG>(P + g0, Po);
    } else {
      dg_ld_line<SEG>(P + g0, Po);
    }
    if (mp.do_cfl) {
#pragma unroll
      for (int m = 0; m < SEG; ++m) {
        const double sp = dg_cfl_speed<EOS, ND>(eos, Uo[m], Po[m], mp.cw);
        if (sp > 0.0) speed = fmax(speed, sp);
      }
    }
  }
  const int slot = (int)((blockIdx.x * 4 + wrp) % DG_NSLOT) * DG_SLOT_STRIDE;
  if (mp.do_cfl) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) speed = fmax(speed, __shfl_xor_sync(0xffffffffu, speed, o));
    if (lane == 0 && speed > 0.0) atomicMax(amax + slot, dg_ord(speed));
  }
  const int nlim = (lim && lt == 0) ? 1 : 0;
  const unsigned any = __ballot_sync(0xffffffffu, (nlim | nfail | nfall) != 0);
  if (any) {
    int c0 = nlim, c1 = nfail, c2 = nfall;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      c0 += __shfl_xor_sync(0xffffffffu, c0, o);
      c1 += __shfl_xor_sync(0xffffffffu, c1, o);
      c2 += __shfl_xor_sync(0xffffffffu, c2, o);
    }
    if (lane == 0 && counters) {                            // NULL: the stand-alone call keeps no counts
      if (c0) atomicAdd(&counters[slot + 4], (dg_ull)c0);
      if (c1) atomicAdd(&counters[slot + 2], (dg_ull)c1);
      if (c2) atomicAdd(&counters[slot + 3], (dg_ull)c2);
    }
  }
}

// FP64 FMA throughput probe (the roofline denominator of the ALU-bound kernels, measured on the box
// instead of derived from unit counts): 8 independent DFMA chains per thread, no memory traffic.
__global__ void __launch_bounds__(256)
dg_fp64_probe_kernel(double* out, int iters, double seed) {
  double x[8];
#pragma unroll
  for (int c = 0; c < 8; ++c) x[c] = seed + 1e-3 * (threadIdx.x + c);
  const double a = 0.999999, b = 1e-7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int c = 0; c < 8; ++c) x[c] = fma(x[c], a, b);
  }
  double sum = 0.0;
#pragma unroll
  for (int c = 0; c < 8; ++c) sum += x[c];
  if (sum == 123.456) out[0] = sum;                 // never true: keeps the chains alive
}

// dt for the coming step, on the device: fixed (dt_fixed > 0) or cfl / amax (reading R11); consumes
// the accumulated maximum (the step's last stage refills it), advances the elapsed time.  A maximum
// that is not a positive finite number (every speed NaN after con2prim failures, an empty state)
// gives dt = 0 -- the step leaves the state unchanged -- and counts one bad step.
__global__ void dg_dt_kernel(double dt_fixed, double cfl, dg_ull* amax, double* dt_out, double* t_acc,
                             dg_ull* n_stages, dg_ull* n_bad_dt, int stages) {
  double m = 0.0;
  for (int s = 0; s < DG_NSLOT; ++s) {
    m = fmax(m, dg_unord(amax[s * DG_SLOT_STRIDE]));
    amax[s * DG_SLOT_STRIDE] = 0ull;
  }
  double dt = dt_fixed;
  if (!(dt_fixed > 0.0)) {
    dt = cfl / m;
    if (!(m > 0.0) || !isfinite(dt)) { dt = 0.0; *n_bad_dt += 1ull; }
  }
  *dt_out = dt;
  *t_acc += dt;
  *n_stages += (dg_ull)stages;
}

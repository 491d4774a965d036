// flat_kernels.cuh -- the point-wise and cell-wise kernels of the CUDA path that need no
// neighbour data (sm_100a, fp64):
//   dg_c2p_batch_kernel    conserved -> primitive over a flat SoA batch
//   dg_p2c_batch_kernel    primitive -> conserved (Eq. 4)
//   dg_c2p_state_kernel    the same recovery on a context state, plus the failure counter and
//                          the CFL wave-speed maximum (reading R11)
//   dg_limiter_kernel      the physicality-enforcing operator on caller data
//   dg_dt_kernel           dt = cfl / amax on the device (no host round trip)
// All are HBM-streaming kernels: one thread per state / node, SoA rows read and written with
// fully coalesced 8-byte accesses (32 lanes x 8 B = one 256 B line per variable per warp).
#pragma once
#include "stage_kernel.cuh"

#define DG_FLAT_NT 256

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

#ifndef DG_C2P_MINB
#define DG_C2P_MINB 6      // 6 x 256 threads per SM (42 registers): best of a 1..8 sweep
#endif
template <int EOS>
__global__ void __launch_bounds__(DG_FLAT_NT, DG_C2P_MINB)
dg_c2p_batch_kernel(long long n, const double* __restrict__ U, double* __restrict__ W,
                    int* __restrict__ status, EosPar eos) {
  const long long i = (long long)blockIdx.x * DG_FLAT_NT + threadIdx.x;
  if (i >= n) return;
  double u[5], w[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) u[v] = __ldg(U + v * n + i);
  const int st = dg_con2prim<EOS>(eos, u, w);
#pragma unroll
  for (int v = 0; v < 5; ++v) W[v * n + i] = w[v];
  if (status) status[i] = st;
}

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

// W = p(U) at every node of a state (Eq. 16); W may be NULL (CFL only).  counters[2] += failures.
// amax (or NULL): atomicMax of sum_d cw[d] max(|lambda-_d|,|lambda+_d|) over the nodes (R11).
template <int EOS, int ND>
__global__ void __launch_bounds__(DG_FLAT_NT)
dg_c2p_state_kernel(long long n, const double* __restrict__ U, double* __restrict__ W, EosPar eos,
                    double cw0, double cw1, double cw2, dg_ull* amax, dg_ull* counters) {
  __shared__ double sRed[32];
  __shared__ int sFail;
  if (threadIdx.x == 0) sFail = 0;
  __syncthreads();
  const long long i = (long long)blockIdx.x * DG_FLAT_NT + threadIdx.x;
  double speed = 0.0;
  if (i < n) {
    double u[5], w[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) u[v] = __ldg(U + v * n + i);
    const int st = dg_con2prim<EOS>(eos, u, w);
    if (W) {
#pragma unroll
      for (int v = 0; v < 5; ++v) W[v * n + i] = w[v];
    }
    if (st != 0) atomicAdd(&sFail, 1);
    if (amax) {
      const double cw[3] = {cw0, cw1, cw2};
      const double s = dg_cfl_speed<EOS, ND>(eos, w, cw);
      if (s > 0.0) speed = s;                       // NaN never wins
    }
  }
  if (amax) dg_block_atomic_max(speed, sRed, amax);
  __syncthreads();
  if (threadIdx.x == 0 && sFail && counters) atomicAdd(&counters[2], (dg_ull)sFail);
}

// The physicality-enforcing operator on a canonical-layout state, NE cells per block, one thread
// per node.  flag[n_e] / s[n_e] optional; counters[0..1] += flagged cells / inadmissible means.
template <int NN>
struct LimShape {
  static constexpr int NE = (256 / NN) > 0 ? (256 / NN) : 1;
  static constexpr int NTN = NE * NN;
  static constexpr int NT = (NTN + 31) / 32 * 32;
};

template <int ND, int N>
__global__ void __launch_bounds__(LimShape<dg_ipow(N, ND)>::NT)
dg_limiter_kernel(long long nelem, long long ndof, double* U, unsigned char* flag, double* s_out,
                  const double* __restrict__ wnode /* [NN] tensor weights */, double wsum,
                  double f_screen, double f_solve, double one_m_delta, dg_ull* counters) {
  constexpr int NN = dg_ipow(N, ND);
  using LS = LimShape<NN>;
  __shared__ double scratch[5 * LS::NTN];
  __shared__ double sMean[5 * LS::NE];
  __shared__ dg_ull sSmin[LS::NE];
  __shared__ int sFlag[LS::NE];
  __shared__ int sCnt[2];
  const int t = threadIdx.x;
  const int le = t / NN, n = t - le * NN;
  const long long e = (long long)blockIdx.x * LS::NE + le;
  const bool active = (t < LS::NTN) && (e < nelem);
  if (t < LS::NE) { sSmin[t] = dg_ord(1.0); sFlag[t] = 0; }
  if (t < 2) sCnt[t] = 0;
  __syncthreads();
  double Uo[5] = {0, 0, 0, 0, 0};
  const long long g = e * NN + n;
  if (active) {
#pragma unroll
    for (int v = 0; v < 5; ++v) Uo[v] = U[v * ndof + g];
  }
  const double wn = active ? wnode[n] : 0.0;
  double s;
  const bool flagged = dg_limiter_block<NN, LS::NE, LS::NTN>(Uo, active, t, le, n, wn, wsum, f_screen,
                                                            f_solve, one_m_delta, scratch, sMean,
                                                            sSmin, sFlag, sCnt, s);
  if (active && flagged) {
#pragma unroll
    for (int v = 0; v < 5; ++v) U[v * ndof + g] = Uo[v];
  }
  if (active && n == 0) {
    if (flag) flag[e] = flagged ? 1 : 0;
    if (s_out) s_out[e] = s;
  }
  __syncthreads();
  if (t == 0 && counters) {
    if (sCnt[0]) atomicAdd(&counters[0], (dg_ull)sCnt[0]);
    if (sCnt[1]) atomicAdd(&counters[1], (dg_ull)sCnt[1]);
  }
}

// dt for the coming step, on the device: fixed (dt_fixed > 0) or cfl / amax (reading R11); consumes
// the accumulated maximum (the step's last stage refills it), advances the elapsed time.
__global__ void dg_dt_kernel(double dt_fixed, double cfl, dg_ull* amax, double* dt_out, double* t_acc,
                             dg_ull* n_stages, int stages) {
  const double m = dg_unord(*amax);
  const double dt = (dt_fixed > 0.0) ? dt_fixed : cfl / m;
  *amax = 0ull;
  *dt_out = dt;
  *t_acc += dt;
  *n_stages += (dg_ull)stages;
}

// dgrhd.cu -- host side of the C ABI declared in include/dgrhd.h: argument checks, the context
// (operator tables, buffer carving inside the caller's workspace, device scalars), kernel
// dispatch and the step orchestration.  No device memory is allocated here; every launch goes to
// the caller's stream; there is no CPU fallback (every compute call needs a CUDA device).
#include "../../include/dgrhd.h"

#include <cmath>
#include <cstdarg>
#include <cstddef>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#include "basis.h"
#include "flat_kernels.cuh"

// launchers of the fused stage kernel, one translation unit per (ndim, EOS): stage_inst.cu
#define DG_DECL(nd, eos, rs)                                                                      \
  cudaError_t dg_launch_stage_##nd##_##eos##rs(int N, const StageArgs& a, cudaStream_t st); \
  cudaError_t dg_prepare_stage_##nd##_##eos##rs(int N);
DG_DECL(1, 0, 0) DG_DECL(1, 1, 0) DG_DECL(2, 0, 0) DG_DECL(2, 1, 0) DG_DECL(3, 0, 0) DG_DECL(3, 1, 0)
DG_DECL(1, 0, 1) DG_DECL(1, 1, 1) DG_DECL(2, 0, 1) DG_DECL(2, 1, 1) DG_DECL(3, 0, 1) DG_DECL(3, 1, 1)
#undef DG_DECL

// launcher of the con2prim comparison variants: c2p_variant.cu (compiled with -fmad=false)
cudaError_t dg_launch_c2p_variant(int eos, long long n, const double* U, double* W, int* status, EosPar e,
                                  int max_iter, cudaStream_t st);

namespace {

thread_local char g_err[512] = "";


constexpr size_t ALIGN = 256;
inline size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

// device scalars at the head of the workspace.  The CFL maximum and the event counters are spread
// over DG_NSLOT slots, 128 bytes apart (one atomic per thread block: a single address would
// serialise them); readers take the maximum / the sum over the slots.
struct DevScalars {
  double dt;          // time step of the step in flight
  double t_acc;       // sum of the steps taken by the current dgrhd_step call
  dg_ull n_stages;    // RK stages executed by dgrhd_step
  dg_ull n_bad_dt;    // steps whose CFL maximum was not a positive finite number (dt = 0)
  dg_ull call_cnt[2]; // per-call counters of dgrhd_enforce_physicality
  dg_ull pad_[10];
  dg_ull amax[DG_NSLOT * DG_SLOT_STRIDE];      // ordered-int images of the CFL maximum of the state
  dg_ull amax_tmp[DG_NSLOT * DG_SLOT_STRIDE];  // same, for dgrhd_cfl_dt on a caller state
  dg_ull counters[DG_NSLOT * DG_SLOT_STRIDE];  // per slot: n_flagged, n_bad_mean, n_c2p_fail, n_tm_fallback, n_shock_limited
};

bool valid_cfg(const dgrhd_config* c) {
  if (!c) return false;
  if (c->ndim < 1 || c->ndim > 3) return false;
  for (int d = 0; d < 3; ++d) {
    if (c->nelem[d] < 1 || c->nelem[d] > 2147483647LL) return false;
    if (d >= c->ndim && c->nelem[d] != 1) return false;
    if (d < c->ndim && !(c->xmax[d] > c->xmin[d])) return false;
    if (d < c->ndim) {                       // bc[d] = lo + 256*hi, hi = 0: same as lo
      const int lo = c->bc[d] & 255, hi = (c->bc[d] >> 8) & 255;
      if (c->bc[d] < 0 || c->bc[d] > 0xffff || lo > DGRHD_BC_DIRICHLET || hi > DGRHD_BC_DIRICHLET) return false;
      if (lo == DGRHD_BC_PERIODIC && hi != 0) return false;     // periodic is both ends
      for (int sd = 0; sd < 2; ++sd) {
        const int k = (sd && hi) ? hi : lo;
        if (k == DGRHD_BC_DIRICHLET) {                          // ghost primitives: finite, rho > 0, P > 0
          const double* w = c->bc_state[d][sd];
          for (int v = 0; v < 5; ++v)
            if (!std::isfinite(w[v])) return false;
          if (!(w[0] > 0.0 && w[4] > 0.0)) return false;
        }
      }
    }
  }
  if (c->riemann != DGRHD_RIEMANN_HLL && c->riemann != DGRHD_RIEMANN_HLLC) return false;
  if (c->shock_limiter != DGRHD_SHOCK_LIMITER_NONE && c->shock_limiter != DGRHD_SHOCK_LIMITER_MOE &&
      c->shock_limiter != DGRHD_SHOCK_LIMITER_MINMOD) return false;
  if (!(c->moe_alpha >= 0.0)) return false;
  if (c->order_p < 0 || c->order_p > 4) return false;
  if (c->eos != DGRHD_EOS_IDEAL && c->eos != DGRHD_EOS_TAUB_MATTHEWS) return false;
  if (c->eos == DGRHD_EOS_IDEAL && !(c->gamma_ad > 1.0)) return false;
  if (c->rk_stages < 1 || c->rk_stages > 3) return false;
  {                                         // kernels index nodes with 32-bit integers
    double nd = 1.0;
    for (int d = 0; d < c->ndim; ++d) nd *= (double)c->nelem[d] * (c->order_p + 1);
    if (nd >= 2147483648.0) return false;
  }
  if (!(c->eps_q >= 0.0 && c->eps_q < 0.5) || !(c->delta_s >= 0.0 && c->delta_s < 0.5)) return false;
  return true;
}

int ipow(int b, int e) { int r = 1; while (e-- > 0) r *= b; return r; }

EosPar make_eos(int eos, double G) {
  EosPar e;
  e.G = G;
  e.al = (eos == DGRHD_EOS_IDEAL) ? G / (G - 1.0) : 0.0;
  return e;
}

}  // namespace

struct dgrhd_ctx {
  dgrhd_config cfg;
  int N, NN;
  long long nelem, ndof;
  size_t state_bytes;
  cudaStream_t stream;
  DevScalars* sc;
  // B[0..2]: state buffers (5 x ndof each); the state lives in B[par] for RK1 (whose output cannot
  // overwrite its input: neighbouring blocks read their halo from it) and in B[0] otherwise.
  // P[0..1]: pressure of the stage input / output, ping-pong; P[par] belongs to the state.
  double* B[3];
  double* P[2];
  double* moe_stats;        // [n_e][15] cell average / maximum / minimum (shock limiter), else NULL
  int par;
  bool has_state;
  BasisTables basis;
  double wsum;
  EosPar eos;
  // one captured CUDA graph per parity: a whole SSP-RK step (dt kernel + stages)
  int use_graph;
  cudaStream_t cap_stream;
  cudaGraphExec_t gexec[2];
  double gdt[2];
  dg_ull bad_dt_seen;       // n_bad_dt as last read back by dgrhd_step / dgrhd_get_counters
  char err[512];
};

static int fail(dgrhd_ctx* c, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (c) snprintf(c->err, sizeof c->err, "%s", buf);
  snprintf(g_err, sizeof g_err, "%s", buf);
  return code;
}

static int cuda_fail(dgrhd_ctx* c, cudaError_t e, const char* where) {
  return fail(c, DGRHD_ECUDA, "%s: %s", where, cudaGetErrorString(e));
}

#define DG_CUDA(c, call)                                  \
  do {                                                    \
    cudaError_t e__ = (call);                             \
    if (e__ != cudaSuccess) return cuda_fail(c, e__, #call); \
  } while (0)

static inline double* state_buf(dgrhd_ctx* c) { return c->B[c->cfg.rk_stages == 1 ? c->par : 0]; }
static inline bool aligned16(const void* p) { return ((uintptr_t)p & 15u) == 0; }

// ------------------------------------------------------------------------------------------------
// kernel dispatch helpers
// ------------------------------------------------------------------------------------------------
#define DG_CASES(FN, ARGS)                                                         \
  switch (c->cfg.ndim * 4 + c->cfg.eos * 2 + c->cfg.riemann) {                     \
    case 4: return dg_##FN##_stage_1_00 ARGS;  case 5: return dg_##FN##_stage_1_01 ARGS;   \
    case 6: return dg_##FN##_stage_1_10 ARGS;  case 7: return dg_##FN##_stage_1_11 ARGS;   \
    case 8: return dg_##FN##_stage_2_00 ARGS;  case 9: return dg_##FN##_stage_2_01 ARGS;   \
    case 10: return dg_##FN##_stage_2_10 ARGS; case 11: return dg_##FN##_stage_2_11 ARGS;  \
    case 12: return dg_##FN##_stage_3_00 ARGS; case 13: return dg_##FN##_stage_3_01 ARGS;  \
    case 14: return dg_##FN##_stage_3_10 ARGS; case 15: return dg_##FN##_stage_3_11 ARGS;  \
  }                                                                                \
  return cudaErrorInvalidValue;

static cudaError_t launch_stage(dgrhd_ctx* c, const StageArgs& a) { DG_CASES(launch, (c->N, a, c->stream)) }
static cudaError_t prepare_stage(dgrhd_ctx* c) { DG_CASES(prepare, (c->N)) }
#undef DG_CASES

// Eq. 4 on the host, for the Dirichlet ghost states: U = [gamma rho, gamma rho h u, gamma^2 rho h - P],
// rho h by Eq. 8 (ideal) or Eq. 10 (Taub-Matthews)
static void host_prim2con(int eos, double G, const double W[5], double U[5]) {
  const double g2 = 1.0 + W[1] * W[1] + W[2] * W[2] + W[3] * W[3], g = std::sqrt(g2);
  const double rh = (eos == DGRHD_EOS_IDEAL) ? W[0] + G / (G - 1.0) * W[4]
                                             : 2.5 * W[4] + 1.5 * std::sqrt(W[4] * W[4] + 4.0 / 9.0 * W[0] * W[0]);
  U[0] = g * W[0];
  for (int k = 1; k <= 3; ++k) U[k] = g * rh * W[k];
  U[4] = g2 * rh - W[4];
}

// P = P(U) over a state (+ all primitives when W != NULL, + failure counts, + CFL maximum when
// amax != NULL)
static cudaError_t launch_c2p_state(dgrhd_ctx* c, const double* U, double* P, double* W, dg_ull* amax,
                                    dg_ull* counters) {
  const long long n = c->ndof;
  const unsigned nb = (unsigned)((n + DG_FLAT_NT - 1) / DG_FLAT_NT);
  double cw[3] = {0, 0, 0};
  for (int d = 0; d < c->cfg.ndim; ++d)
    cw[d] = (2.0 * c->cfg.order_p + 1.0) * (double)c->cfg.nelem[d] / (c->cfg.xmax[d] - c->cfg.xmin[d]);
#define DG_GO(E, D) \
  dg_c2p_state_kernel<E, D><<<nb, DG_FLAT_NT, 0, c->stream>>>(n, U, P, W, c->eos, cw[0], cw[1], cw[2], amax, counters)
  if (c->cfg.eos == DGRHD_EOS_IDEAL) {
    if (c->cfg.ndim == 1) DG_GO(0, 1); else if (c->cfg.ndim == 2) DG_GO(0, 2); else DG_GO(0, 3);
  } else {
    if (c->cfg.ndim == 1) DG_GO(1, 1); else if (c->cfg.ndim == 2) DG_GO(1, 2); else DG_GO(1, 3);
  }
#undef DG_GO
  return cudaGetLastError();
}

static LimPar make_limpar(dgrhd_ctx* c) {
  LimPar lp;
  for (int i = 0; i < 5; ++i) lp.w[i] = (i < c->N) ? c->basis.w[i] : 0.0;
  lp.wsum = c->wsum;
  lp.f_screen = 1.0 - 0.5 * c->cfg.eps_q;
  lp.f_solve = 1.0 - c->cfg.eps_q;
  lp.one_m_delta = 1.0 - c->cfg.delta_s;
  return lp;
}

template <int ND>
static cudaError_t launch_limiter_nd(dgrhd_ctx* c, double* U, unsigned char* flag, double* s,
                                     dg_ull* counters) {
  const LimPar lp = make_limpar(c);
#define DG_GO(NV)                                                                                  \
  {                                                                                                \
    constexpr int EPB = 4 * TileShape<ND, NV>::EPW;                                                \
    const unsigned nb = (unsigned)((c->nelem + EPB - 1) / EPB);                                    \
    dg_limiter_kernel<ND, NV><<<nb, 128, 0, c->stream>>>(c->nelem, c->ndof, U, flag, s, lp, counters); \
  }
  switch (c->N) {
    case 1: DG_GO(1) break;
    case 2: DG_GO(2) break;
    case 3: DG_GO(3) break;
    case 4: DG_GO(4) break;
    case 5: DG_GO(5) break;
  }
#undef DG_GO
  return cudaGetLastError();
}

static cudaError_t launch_limiter(dgrhd_ctx* c, double* U, unsigned char* flag, double* s,
                                  dg_ull* counters) {
  if (c->cfg.ndim == 1) return launch_limiter_nd<1>(c, U, flag, s, counters);
  if (c->cfg.ndim == 2) return launch_limiter_nd<2>(c, U, flag, s, counters);
  return launch_limiter_nd<3>(c, U, flag, s, counters);
}

// The shock limiter on a stage's output (U, P): cell statistics, then bounds / theta / rescale, the
// pressure of the rescaled cells and, on the step's last stage, the CFL maximum of the limited state.
template <int ND>
static cudaError_t launch_moe_nd(dgrhd_ctx* c, double* U, double* P, int do_cfl, dg_ull* amax, dg_ull* counters,
                                 double* theta) {
  const LimPar lp = make_limpar(c);
  MoePar mp;
  for (int d = 0; d < 3; ++d) {
    mp.ne[d] = c->cfg.nelem[d];
    mp.periodic[d] = (d < c->cfg.ndim && (c->cfg.bc[d] & 255) == DGRHD_BC_PERIODIC) ? 1 : 0;
    mp.cw[d] = (d < c->cfg.ndim) ? (2.0 * c->cfg.order_p + 1.0) * (double)c->cfg.nelem[d] / (c->cfg.xmax[d] - c->cfg.xmin[d]) : 0.0;
  }
  const bool minmod = (c->cfg.shock_limiter == DGRHD_SHOCK_LIMITER_MINMOD);
  mp.alpha = minmod ? (c->cfg.moe_alpha > 0.0 ? c->cfg.moe_alpha : 1.0) : c->cfg.moe_alpha;
  MmPar mm;
  {
    double sxx = 0.0, sw = 0.0;
    for (int i = 0; i < 5; ++i) mm.x[i] = (i < c->N) ? c->basis.x[i] : 0.0;
    for (int i = 0; i < c->N; ++i) { sxx += c->basis.w[i] * c->basis.x[i] * c->basis.x[i]; sw += c->basis.w[i]; }
    for (int d = 1; d < c->cfg.ndim; ++d) sxx *= sw;
    mm.rxx = (sxx > 0.0) ? 1.0 / sxx : 0.0;
  }
  mp.do_cfl = do_cfl;
#define DG_GO(NV)                                                                                       \
  {                                                                                                     \
    constexpr int EPB = 4 * TileShape<ND, NV>::EPW;                                                     \
    const unsigned nb = (unsigned)((c->nelem + EPB - 1) / EPB);                                         \
    if (minmod)                                                                                         \
      dg_mm_stats_kernel<ND, NV><<<nb, 128, 0, c->stream>>>(c->nelem, c->ndof, U, c->moe_stats, lp, mm); \
    else                                                                                                \
      dg_moe_stats_kernel<ND, NV><<<nb, 128, 0, c->stream>>>(c->nelem, c->ndof, U, c->moe_stats, lp);   \
    if (c->cfg.eos == DGRHD_EOS_IDEAL) {                                                                \
      if (minmod) dg_moe_apply_kernel<ND, NV, 0, 1><<<nb, 128, 0, c->stream>>>(c->nelem, c->ndof, U, P, c->moe_stats, mp, c->eos, amax, counters, theta); \
      else dg_moe_apply_kernel<ND, NV, 0, 0><<<nb, 128, 0, c->stream>>>(c->nelem, c->ndof, U, P, c->moe_stats, mp, c->eos, amax, counters, theta); \
    } else {                                                                                            \
      if (minmod) dg_moe_apply_kernel<ND, NV, 1, 1><<<nb, 128, 0, c->stream>>>(c->nelem, c->ndof, U, P, c->moe_stats, mp, c->eos, amax, counters, theta); \
      else dg_moe_apply_kernel<ND, NV, 1, 0><<<nb, 128, 0, c->stream>>>(c->nelem, c->ndof, U, P, c->moe_stats, mp, c->eos, amax, counters, theta); \
    }                                                                                                   \
  }
  switch (c->N) {
    case 1: DG_GO(1) break;
    case 2: DG_GO(2) break;
    case 3: DG_GO(3) break;
    case 4: DG_GO(4) break;
    case 5: DG_GO(5) break;
  }
#undef DG_GO
  return cudaGetLastError();
}

static cudaError_t launch_moe(dgrhd_ctx* c, double* U, double* P, int do_cfl, dg_ull* amax, dg_ull* counters,
                              double* theta) {
  if (c->cfg.ndim == 1) return launch_moe_nd<1>(c, U, P, do_cfl, amax, counters, theta);
  if (c->cfg.ndim == 2) return launch_moe_nd<2>(c, U, P, do_cfl, amax, counters, theta);
  return launch_moe_nd<3>(c, U, P, do_cfl, amax, counters, theta);
}

static void fill_stage_args(dgrhd_ctx* c, StageArgs& a) {
  memset(&a, 0, sizeof a);
  a.ndof = c->ndof;
  const int N = c->N;
  for (int d = 0; d < 3; ++d) {
    a.ne[d] = (int)c->cfg.nelem[d];
    if (d < c->cfg.ndim) {
      const double h = (c->cfg.xmax[d] - c->cfg.xmin[d]) / (double)c->cfg.nelem[d];
      const double rh = 2.0 / h;
      a.cw[d] = (2.0 * c->cfg.order_p + 1.0) * (double)c->cfg.nelem[d] / (c->cfg.xmax[d] - c->cfg.xmin[d]);
      a.lift[d] = rh * c->basis.lift;
      double* D = (d == 0) ? a.Dx : (d == 1 ? a.Dy : a.Dz);
      for (int i = 0; i < N; ++i)
        for (int q = 0; q < N; ++q) D[i * N + q] = rh * c->basis.Dhat[i][q];
    }
  }
  a.f_screen = 1.0 - 0.5 * c->cfg.eps_q;
  a.f_solve = 1.0 - c->cfg.eps_q;
  a.one_m_delta = 1.0 - c->cfg.delta_s;
  a.eos = c->eos;
  a.dt_ptr = &c->sc->dt;
  a.amax = c->sc->amax;
  a.counters = c->sc->counters;
  for (int i = 0; i < N; ++i) a.w[i] = c->basis.w[i];
  // halo offsets: the node facing a boundary node of a tile lies one element over (interior), or, on
  // the first / last tile of the axis, in the element at the other end (periodic) / is the node
  // itself (outflow, reading R12)
  {
    const int NN = c->NN;
    const long long es[3] = {1, c->cfg.nelem[0], c->cfg.nelem[0] * c->cfg.nelem[1]};
    int sn = 1;
    for (int d = 0; d < 3; ++d, sn *= N) {
      const long long step = es[d] * NN, layer = (long long)(N - 1) * sn;
      a.hoff[d][0] = (int)(-step + layer);                 // minus side: neighbour e-1, node layer N-1
      a.hoff[d][1] = (int)(step - layer);                  // plus side:  neighbour e+1, node layer 0
      const int lo = c->cfg.bc[d] & 255, hi = (c->cfg.bc[d] >> 8) & 255;
      if (d < c->cfg.ndim && lo == DGRHD_BC_PERIODIC) {
        a.hfix[d][0] = (int)(c->cfg.nelem[d] * step);      // e-1 -> e-1+ne
        a.hfix[d][1] = (int)(-c->cfg.nelem[d] * step);
      } else {                                             // own node: total offset 0; the ghost state
        a.hfix[d][0] = -a.hoff[d][0];                      // is made from it (outflow: as is, wall:
        a.hfix[d][1] = -a.hoff[d][1];                      // normal momentum reversed) or replaced
        for (int sd = 0; sd < 2 && d < c->cfg.ndim; ++sd) {
          const int k = (sd && hi) ? hi : lo;
          a.bcm[d][sd] = (k == DGRHD_BC_REFLECT || k == DGRHD_BC_DIRICHLET) ? k : 0;
          if (k == DGRHD_BC_DIRICHLET) {
            host_prim2con(c->cfg.eos, c->cfg.gamma_ad, c->cfg.bc_state[d][sd], a.bcU[d][sd]);
            a.bcU[d][sd][5] = c->cfg.bc_state[d][sd][4];
          }
        }
      }
    }
  }
  a.wsum = c->wsum;
}

// ------------------------------------------------------------------------------------------------
// create / destroy
// ------------------------------------------------------------------------------------------------
static size_t pbuf_bytes(long long ndof) { return align_up((size_t)ndof * sizeof(double)); }
static size_t moe_bytes(const dgrhd_config* cfg, long long ne) {
  return cfg->shock_limiter ? align_up((size_t)ne * 25 * sizeof(double)) : 0;   // Moe uses 15, minmod 25 per cell
}

extern "C" size_t dgrhd_workspace_bytes(const dgrhd_config* cfg) {
  if (!valid_cfg(cfg)) return 0;
  long long ne = 1;
  for (int d = 0; d < cfg->ndim; ++d) ne *= cfg->nelem[d];
  const long long ndof = ne * ipow(cfg->order_p + 1, cfg->ndim);
  const size_t sb = align_up((size_t)ndof * 5 * sizeof(double));
  return align_up(sizeof(DevScalars)) + 3 * sb + 2 * pbuf_bytes(ndof) + moe_bytes(cfg, ne);
}

extern "C" int dgrhd_create(const dgrhd_config* cfg, void* workspace_dev, size_t workspace_bytes,
                            void* cuda_stream, dgrhd_ctx** out) {
  if (out) *out = nullptr;
  if (!out || !valid_cfg(cfg)) return fail(nullptr, DGRHD_EINVAL, "dgrhd_create: invalid configuration");
  if (!workspace_dev || ((uintptr_t)workspace_dev % ALIGN) != 0)
    return fail(nullptr, DGRHD_EINVAL, "dgrhd_create: workspace NULL or not 256-byte aligned");
  const size_t need = dgrhd_workspace_bytes(cfg);
  if (workspace_bytes < need)
    return fail(nullptr, DGRHD_ENOMEM, "dgrhd_create: workspace %zu < %zu bytes", workspace_bytes, need);
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
    return fail(nullptr, DGRHD_ECUDA, "dgrhd_create: no CUDA device (there is no CPU fallback)");
  dgrhd_ctx* c = new (std::nothrow) dgrhd_ctx;
  if (!c) return fail(nullptr, DGRHD_ENOMEM, "dgrhd_create: host allocation failed");
  memset(c, 0, sizeof *c);
  c->cfg = *cfg;
  c->N = cfg->order_p + 1;
  c->NN = ipow(c->N, cfg->ndim);
  c->nelem = 1;
  for (int d = 0; d < cfg->ndim; ++d) c->nelem *= cfg->nelem[d];
  c->ndof = c->nelem * c->NN;
  c->state_bytes = (size_t)c->ndof * 5 * sizeof(double);
  c->stream = (cudaStream_t)cuda_stream;
  c->eos = make_eos(cfg->eos, cfg->gamma_ad);
  dgbasis::build(c->N, c->basis);
  char* p = (char*)workspace_dev;
  c->sc = (DevScalars*)p;  p += align_up(sizeof(DevScalars));
  const size_t sb = align_up(c->state_bytes);
  for (int i = 0; i < 3; ++i) { c->B[i] = (double*)p;  p += sb; }
  for (int i = 0; i < 2; ++i) { c->P[i] = (double*)p;  p += pbuf_bytes(c->ndof); }
  c->moe_stats = cfg->shock_limiter ? (double*)p : nullptr;
  // sum of the tensor weights (summed in node order)
  c->wsum = 0.0;
  for (int n = 0; n < c->NN; ++n) {
    double w = c->basis.w[n % c->N];
    if (cfg->ndim > 1) w *= c->basis.w[(n / c->N) % c->N];
    if (cfg->ndim > 2) w *= c->basis.w[n / (c->N * c->N)];
    c->wsum += w;
  }
  // per-device kernel attributes (shared-memory opt-in) for this context's instantiation, outside
  // any stream capture
  cudaError_t e = prepare_stage(c);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->sc, 0, sizeof(DevScalars), c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) {
    int r = cuda_fail(nullptr, e, "dgrhd_create");
    delete c;
    return r;
  }
  c->use_graph = (cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) == cudaSuccess) ? 1 : 0;
  *out = c;
  return DGRHD_OK;
}

extern "C" int dgrhd_set_option(dgrhd_ctx* c, int option, int value) {
  if (!c) return DGRHD_EINVAL;
  if (option == DGRHD_OPT_CUDA_GRAPH) {
    c->use_graph = (value != 0 && c->cap_stream) ? 1 : 0;
    return DGRHD_OK;
  }
  return fail(c, DGRHD_EINVAL, "dgrhd_set_option: unknown option %d", option);
}

extern "C" int dgrhd_destroy(dgrhd_ctx* ctx) {
  if (!ctx) return DGRHD_EINVAL;
  for (int i = 0; i < 2; ++i)
    if (ctx->gexec[i]) cudaGraphExecDestroy(ctx->gexec[i]);
  if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
  delete ctx;
  return DGRHD_OK;
}

// ------------------------------------------------------------------------------------------------
// state access
// ------------------------------------------------------------------------------------------------
static int refresh_state_pressure(dgrhd_ctx* c) {
  DG_CUDA(c, cudaMemsetAsync(c->sc->amax, 0, sizeof c->sc->amax, c->stream));
  DG_CUDA(c, launch_c2p_state(c, state_buf(c), c->P[c->par], nullptr, c->sc->amax, c->sc->counters));
  return DGRHD_OK;
}

extern "C" int dgrhd_set_state(dgrhd_ctx* c, const double* U_dev) {
  if (!c || !U_dev) return fail(c, DGRHD_EINVAL, "dgrhd_set_state: NULL argument");
  c->par = 0;
  DG_CUDA(c, cudaMemcpyAsync(c->B[0], U_dev, c->state_bytes, cudaMemcpyDeviceToDevice, c->stream));
  const int r = refresh_state_pressure(c);
  if (r != DGRHD_OK) return r;
  c->has_state = true;
  return DGRHD_OK;
}

extern "C" int dgrhd_get_state(dgrhd_ctx* c, double* U_dev) {
  if (!c || !U_dev) return fail(c, DGRHD_EINVAL, "dgrhd_get_state: NULL argument");
  if (!c->has_state) return fail(c, DGRHD_ESTATE, "dgrhd_get_state: no state set");
  DG_CUDA(c, cudaMemcpyAsync(U_dev, state_buf(c), c->state_bytes, cudaMemcpyDeviceToDevice, c->stream));
  return DGRHD_OK;
}

extern "C" int dgrhd_get_prims(dgrhd_ctx* c, double* W_dev) {
  if (!c || !W_dev) return fail(c, DGRHD_EINVAL, "dgrhd_get_prims: NULL argument");
  if (!c->has_state) return fail(c, DGRHD_ESTATE, "dgrhd_get_prims: no state set");
  DG_CUDA(c, launch_c2p_state(c, state_buf(c), nullptr, W_dev, nullptr, nullptr));
  return DGRHD_OK;
}

// ------------------------------------------------------------------------------------------------
// R = L(U) on caller buffers: nodal pressure into the spare pressure buffer, then the fused kernel
// in MODE_RHS
// ------------------------------------------------------------------------------------------------
extern "C" int dgrhd_rhs(dgrhd_ctx* c, const double* U_dev, double* R_dev) {
  if (!c || !U_dev || !R_dev) return fail(c, DGRHD_EINVAL, "dgrhd_rhs: NULL argument");
  if (U_dev == R_dev) return fail(c, DGRHD_EINVAL, "dgrhd_rhs: U_dev and R_dev overlap");
  if (!aligned16(U_dev) || !aligned16(R_dev))
    return fail(c, DGRHD_EINVAL, "dgrhd_rhs: state pointers must be 16-byte aligned");
  double* Ptmp = c->P[c->par ^ 1];
  DG_CUDA(c, launch_c2p_state(c, U_dev, Ptmp, nullptr, nullptr, c->sc->counters));
  StageArgs a;
  fill_stage_args(c, a);
  a.mode = DG_MODE_RHS;
  a.Us = U_dev;
  a.Pin = Ptmp;
  a.Rout = R_dev;
  DG_CUDA(c, launch_stage(c, a));
  return DGRHD_OK;
}

// ------------------------------------------------------------------------------------------------
// R = L(U) without a context or a workspace (dgrhd_rhs_static, include/dgrhd.h): for callers that
// cannot obtain device memory.  Same two kernels as dgrhd_rhs; their scratch -- the device scalars
// (of which MODE_RHS touches only the counter slots) followed by the nodal pressure -- is the array
// below, which every GPU that loads this translation unit's code holds until the process exits.
//
// In host code the name g_rhs_static_scratch is a handle for the runtime's symbol calls, NOT a device
// address: handing it to a kernel would fault or, where the GPU can reach host memory, quietly use the
// wrong memory.  The device address comes from cudaGetSymbolAddress, asked once per device with that
// device current (each device has its own copy of the array), under a mutex, and cached.
// ------------------------------------------------------------------------------------------------
namespace {
constexpr size_t STATIC_HEAD_BYTES = (sizeof(DevScalars) + ALIGN - 1) / ALIGN * ALIGN;
static_assert(STATIC_HEAD_BYTES == 12544, "include/dgrhd.h states this size");
static_assert(STATIC_HEAD_BYTES % sizeof(double) == 0, "the pressure rows follow the head");
constexpr size_t STATIC_WORDS = STATIC_HEAD_BYTES / sizeof(double) + (size_t)DGRHD_STATIC_MAX_NDOF;
constexpr int STATIC_MAX_DEVICES = 64;
}  // namespace

static __device__ __align__(256) double g_rhs_static_scratch[STATIC_WORDS];

namespace {
std::mutex g_static_mu;
double* g_static_addr[STATIC_MAX_DEVICES];                 // device address of the array, per device
unsigned g_static_prepared[STATIC_MAX_DEVICES][6];         // [device][N]: bit (ndim*4 + eos*2 + riemann)
}  // namespace

// One-time set-up per device (and per kernel instantiation): the array's device address and the stage
// kernel's shared-memory opt-in.  Runs with the caller's device current; allocates nothing.
static int static_setup(dgrhd_ctx* c, double** scratch) {
  int dev = -1;
  DG_CUDA(nullptr, cudaGetDevice(&dev));
  if (dev < 0 || dev >= STATIC_MAX_DEVICES)
    return fail(nullptr, DGRHD_ECUDA, "dgrhd_rhs_static: device ordinal %d outside 0..%d", dev, STATIC_MAX_DEVICES - 1);
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_addr[dev]) {
    double* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_rhs_static_scratch);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "dgrhd_rhs_static: cudaGetSymbolAddress");
    if (!p || ((uintptr_t)p % ALIGN) != 0)
      return fail(nullptr, DGRHD_ECUDA, "dgrhd_rhs_static: the built-in scratch array has no usable device address");
    g_static_addr[dev] = p;
  }
  const unsigned bit = 1u << (c->cfg.ndim * 4 + c->cfg.eos * 2 + c->cfg.riemann);
  if (!(g_static_prepared[dev][c->N] & bit)) {
    const cudaError_t e = prepare_stage(c);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "dgrhd_rhs_static: kernel attributes");
    g_static_prepared[dev][c->N] |= bit;
  }
  *scratch = g_static_addr[dev];
  return DGRHD_OK;
}

extern "C" int dgrhd_rhs_static(const dgrhd_config* cfg, const double* U_dev, double* R_dev,
                                int64_t* n_c2p_fail_host, void* cuda_stream) {
  if (!valid_cfg(cfg)) return fail(nullptr, DGRHD_EINVAL, "dgrhd_rhs_static: invalid configuration");
  if (!U_dev || !R_dev) return fail(nullptr, DGRHD_EINVAL, "dgrhd_rhs_static: NULL argument");
  if (U_dev == R_dev) return fail(nullptr, DGRHD_EINVAL, "dgrhd_rhs_static: U_dev and R_dev overlap");
  if (!aligned16(U_dev) || !aligned16(R_dev))
    return fail(nullptr, DGRHD_EINVAL, "dgrhd_rhs_static: state pointers must be 16-byte aligned");
  // a context on the host stack: the host-side fields the launch helpers read, nothing on the device
  dgrhd_ctx c;
  memset(&c, 0, sizeof c);
  c.cfg = *cfg;
  c.N = cfg->order_p + 1;
  c.NN = ipow(c.N, cfg->ndim);
  c.nelem = 1;
  for (int d = 0; d < cfg->ndim; ++d) c.nelem *= cfg->nelem[d];
  c.ndof = c.nelem * c.NN;
  if (c.ndof > (long long)DGRHD_STATIC_MAX_NDOF)
    return fail(nullptr, DGRHD_ENOMEM,
                "dgrhd_rhs_static: the mesh has %lld nodes, the built-in scratch array holds at most %d "
                "(DGRHD_STATIC_MAX_NDOF); use dgrhd_rhs with a workspace of your own for larger meshes",
                c.ndof, (int)DGRHD_STATIC_MAX_NDOF);
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
    return fail(nullptr, DGRHD_ECUDA, "dgrhd_rhs_static: no CUDA device (there is no CPU fallback)");
  c.state_bytes = (size_t)c.ndof * 5 * sizeof(double);
  c.stream = (cudaStream_t)cuda_stream;
  c.eos = make_eos(cfg->eos, cfg->gamma_ad);
  dgbasis::build(c.N, c.basis);
  for (int n = 0; n < c.NN; ++n) {                         // tensor-weight sum, as dgrhd_create forms it
    double w = c.basis.w[n % c.N];
    if (cfg->ndim > 1) w *= c.basis.w[(n / c.N) % c.N];
    if (cfg->ndim > 2) w *= c.basis.w[n / (c.N * c.N)];
    c.wsum += w;
  }
  double* scratch = nullptr;
  const int r = static_setup(&c, &scratch);
  if (r != DGRHD_OK) return r;
  c.sc = (DevScalars*)scratch;
  double* P = scratch + STATIC_HEAD_BYTES / sizeof(double);
  // the array keeps the previous call's contents: the counters must start at zero (the pressure needs
  // no clearing, the first kernel writes all ndof values before the second reads any)
  DG_CUDA(nullptr, cudaMemsetAsync(c.sc, 0, sizeof(DevScalars), c.stream));
  DG_CUDA(nullptr, launch_c2p_state(&c, U_dev, P, nullptr, nullptr, c.sc->counters));
  StageArgs a;
  fill_stage_args(&c, a);
  a.mode = DG_MODE_RHS;
  a.Us = U_dev;
  a.Pin = P;
  a.Rout = R_dev;
  DG_CUDA(nullptr, launch_stage(&c, a));
  if (n_c2p_fail_host) {
    dg_ull h[DG_NSLOT * DG_SLOT_STRIDE];
    DG_CUDA(nullptr, cudaMemcpyAsync(h, c.sc->counters, sizeof h, cudaMemcpyDeviceToHost, c.stream));
    DG_CUDA(nullptr, cudaStreamSynchronize(c.stream));
    dg_ull nfail = 0;
    for (int s = 0; s < DG_NSLOT; ++s) nfail += h[s * DG_SLOT_STRIDE + 2];
    *n_c2p_fail_host = (int64_t)nfail;
  }
  return DGRHD_OK;
}

extern "C" int dgrhd_enforce_physicality(dgrhd_ctx* c, double* U_dev, unsigned char* flag_dev,
                                         double* s_dev, int64_t counters_host[2]) {
  if (!c) return fail(c, DGRHD_EINVAL, "dgrhd_enforce_physicality: NULL context");
  const bool internal = (U_dev == nullptr);
  if (internal && !c->has_state) return fail(c, DGRHD_ESTATE, "dgrhd_enforce_physicality: no state set");
  if (!internal && !aligned16(U_dev))
    return fail(c, DGRHD_EINVAL, "dgrhd_enforce_physicality: state pointer must be 16-byte aligned");
  double* U = internal ? state_buf(c) : U_dev;
  DG_CUDA(c, cudaMemsetAsync(c->sc->call_cnt, 0, 2 * sizeof(dg_ull), c->stream));
  DG_CUDA(c, launch_limiter(c, U, flag_dev, s_dev, c->sc->call_cnt));
  if (internal) {                       // refresh the pressure and the CFL maximum of the state
    const int r = refresh_state_pressure(c);
    if (r != DGRHD_OK) return r;
  }
  if (counters_host) {
    dg_ull h[2];
    DG_CUDA(c, cudaMemcpyAsync(h, c->sc->call_cnt, sizeof h, cudaMemcpyDeviceToHost, c->stream));
    DG_CUDA(c, cudaStreamSynchronize(c->stream));
    counters_host[0] = (int64_t)h[0];
    counters_host[1] = (int64_t)h[1];
  }
  return DGRHD_OK;
}

extern "C" int dgrhd_shock_limiter(dgrhd_ctx* c, double* U_dev, double* theta_dev) {
  if (!c || !U_dev) return fail(c, DGRHD_EINVAL, "dgrhd_shock_limiter: NULL argument");
  if (c->cfg.shock_limiter == DGRHD_SHOCK_LIMITER_NONE)
    return fail(c, DGRHD_ESTATE, "dgrhd_shock_limiter: the context was created without a shock limiter");
  if (!aligned16(U_dev)) return fail(c, DGRHD_EINVAL, "dgrhd_shock_limiter: state pointer must be 16-byte aligned");
  // (the pressure of the rescaled cells lands in the spare pressure buffer; no counters, no CFL: the
  // apply kernel skips both, so neither array is touched)
  DG_CUDA(c, launch_moe(c, U_dev, c->P[c->par ^ 1], 0, nullptr, nullptr, theta_dev));
  return DGRHD_OK;
}

extern "C" int dgrhd_cfl_dt(dgrhd_ctx* c, const double* U_dev, double cfl, double* dt_host) {
  if (!c || !dt_host) return fail(c, DGRHD_EINVAL, "dgrhd_cfl_dt: NULL argument");
  if (!(cfl > 0.0)) return fail(c, DGRHD_EINVAL, "dgrhd_cfl_dt: cfl must be > 0");
  dg_ull* slots = c->sc->amax;
  if (U_dev) {
    slots = c->sc->amax_tmp;
    DG_CUDA(c, cudaMemsetAsync(slots, 0, sizeof c->sc->amax_tmp, c->stream));
    DG_CUDA(c, launch_c2p_state(c, U_dev, nullptr, nullptr, slots, nullptr));
  } else if (!c->has_state) {
    return fail(c, DGRHD_ESTATE, "dgrhd_cfl_dt: no state set");
  }
  static_assert(sizeof(double) == sizeof(dg_ull), "ordered-integer image");
  double h[DG_NSLOT * DG_SLOT_STRIDE];
  DG_CUDA(c, cudaMemcpyAsync(h, slots, sizeof h, cudaMemcpyDeviceToHost, c->stream));
  DG_CUDA(c, cudaStreamSynchronize(c->stream));
  double m = 0.0;
  for (int s = 0; s < DG_NSLOT; ++s)
    if (h[s * DG_SLOT_STRIDE] > m) m = h[s * DG_SLOT_STRIDE];
  const double dt = cfl / m;
  if (!(m > 0.0) || !std::isfinite(dt))
    return fail(c, DGRHD_ESTATE, "dgrhd_cfl_dt: no positive finite wave speed in the state (con2prim failures?)");
  *dt_host = dt;
  return DGRHD_OK;
}

// ------------------------------------------------------------------------------------------------
// SSP-RK steps (Shu-Osher form, reading R10): per step one dt kernel + one fused kernel per stage,
// all on the context's stream, dt and the CFL maximum resident on the device.  A stage's output
// never overwrites its input (other blocks read their halo from it); it may overwrite U0 (each
// thread reads and writes its own nodes only):
//   RK1     B[par] -> B[par^1]
//   SSPRK2  B0 -> B1;  (B1, U0 = B0) -> B0
//   SSPRK3  B0 -> B1;  (B1, U0 = B0) -> B2;  (B2, U0 = B0) -> B0
// The pressure buffers alternate every stage: P[par] -> P[par^1].
// ------------------------------------------------------------------------------------------------
static int enqueue_step(dgrhd_ctx* c, double dt, StageArgs& a) {
  const int S = c->cfg.rk_stages;
  static const double A3[3] = {0.0, 0.75, 1.0 / 3.0}, B3[3] = {1.0, 0.25, 2.0 / 3.0};
  static const double A2[2] = {0.0, 0.5}, B2[2] = {1.0, 0.5};
  dg_dt_kernel<<<1, 1, 0, c->stream>>>(dt, -dt, c->sc->amax, &c->sc->dt, &c->sc->t_acc,
                                       &c->sc->n_stages, &c->sc->n_bad_dt, S);
  DG_CUDA(c, cudaGetLastError());
  for (int s = 0; s < S; ++s) {
    const bool last = (s == S - 1);
    a.a = (S == 2) ? A2[s] : A3[s];
    a.b = (S == 2) ? B2[s] : B3[s];
    if (S == 1) {
      a.Us = c->B[c->par];
      a.Uout = c->B[c->par ^ 1];
      a.U0 = a.Us;
    } else {
      a.Us = c->B[s];
      a.U0 = c->B[0];
      a.Uout = last ? c->B[0] : c->B[s + 1];
    }
    a.Pin = c->P[c->par];
    a.Pout = c->P[c->par ^ 1];
    const bool moe = (c->cfg.shock_limiter != DGRHD_SHOCK_LIMITER_NONE);
    a.do_cfl = (last && !moe) ? 1 : 0;                     // with the shock limiter: taken from the limited state
    DG_CUDA(c, launch_stage(c, a));
    if (moe) DG_CUDA(c, launch_moe(c, a.Uout, a.Pout, last ? 1 : 0, c->sc->amax, c->sc->counters, nullptr));
    c->par ^= 1;
  }
  return DGRHD_OK;
}

// One step through a captured graph (one launch instead of 1 + stages; PAPER.md:755-757 names launch
// overhead as the GPU bottleneck).  The graph is captured on the context's private stream and
// replayed on the caller's stream; it is re-captured when dt (a kernel argument) changes.  Any
// capture failure switches the context back to plain launches.
static int launch_step_graph(dgrhd_ctx* c, double dt, StageArgs& a) {
  const int par = c->par;
  if (!c->gexec[par] || c->gdt[par] != dt) {
    if (c->gexec[par]) { cudaGraphExecDestroy(c->gexec[par]); c->gexec[par] = nullptr; }
    cudaStream_t user = c->stream;
    cudaGraph_t graph = nullptr;
    bool ok = cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
    if (ok) {
      c->stream = c->cap_stream;
      const int r = enqueue_step(c, dt, a);
      c->stream = user;
      c->par = par;
      const cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
      ok = (r == DGRHD_OK) && (e == cudaSuccess) && graph;
    }
    if (ok) ok = cudaGraphInstantiate(&c->gexec[par], graph, 0) == cudaSuccess;
    if (graph) cudaGraphDestroy(graph);
    if (!ok) {
      cudaGetLastError();
      c->gexec[par] = nullptr;
      c->use_graph = 0;
      return enqueue_step(c, dt, a);
    }
    c->gdt[par] = dt;
  }
  DG_CUDA(c, cudaGraphLaunch(c->gexec[par], c->stream));
  c->par = par ^ (c->cfg.rk_stages & 1);
  return DGRHD_OK;
}

extern "C" int dgrhd_step(dgrhd_ctx* c, double dt, int nsteps, double* t_inout_host) {
  if (!c) return fail(c, DGRHD_EINVAL, "dgrhd_step: NULL context");
  if (nsteps < 0 || !(dt == dt)) return fail(c, DGRHD_EINVAL, "dgrhd_step: bad nsteps or dt");
  if (dt == 0.0) return fail(c, DGRHD_EINVAL, "dgrhd_step: dt must be > 0 (fixed) or < 0 (-CFL)");
  if (!c->has_state) return fail(c, DGRHD_ESTATE, "dgrhd_step: no state set");
  DG_CUDA(c, cudaMemsetAsync(&c->sc->t_acc, 0, sizeof(double), c->stream));
  StageArgs a;
  fill_stage_args(c, a);
  a.mode = DG_MODE_STAGE;
  for (int i = 0; i < nsteps; ++i) {
    int r = c->use_graph ? launch_step_graph(c, dt, a) : enqueue_step(c, dt, a);
    if (r != DGRHD_OK) return r;
  }
  if (t_inout_host) {
    struct { double t_acc; dg_ull n_stages, n_bad_dt; } h = {0.0, 0ull, 0ull};   // consecutive in DevScalars
    static_assert(offsetof(DevScalars, n_bad_dt) == offsetof(DevScalars, t_acc) + 16, "read back as one block");
    DG_CUDA(c, cudaMemcpyAsync(&h, &c->sc->t_acc, sizeof h, cudaMemcpyDeviceToHost, c->stream));
    DG_CUDA(c, cudaStreamSynchronize(c->stream));
    *t_inout_host += h.t_acc;
    if (h.n_bad_dt > c->bad_dt_seen) {       // a caller looping to a final time must not spin on dt = 0
      const dg_ull nbad = h.n_bad_dt - c->bad_dt_seen;
      c->bad_dt_seen = h.n_bad_dt;
      return fail(c, DGRHD_ESTATE, "dgrhd_step: %llu step(s) found no positive finite wave speed in the state and "
                  "ran with dt = 0 (con2prim failures? see dgrhd_get_counters)", nbad);
    }
  }
  return DGRHD_OK;
}

extern "C" int dgrhd_run_host(dgrhd_ctx* c, const double* U_host_in, double* U_host_out, double dt,
                              int nsteps, double* t_inout_host) {
  if (!c || !U_host_in || !U_host_out) return fail(c, DGRHD_EINVAL, "dgrhd_run_host: NULL argument");
  c->par = 0;
  DG_CUDA(c, cudaMemcpyAsync(c->B[0], U_host_in, c->state_bytes, cudaMemcpyHostToDevice, c->stream));
  int r = refresh_state_pressure(c);
  if (r != DGRHD_OK) return r;
  c->has_state = true;
  r = dgrhd_step(c, dt, nsteps, nullptr);
  if (r != DGRHD_OK) return r;
  DG_CUDA(c, cudaMemcpyAsync(U_host_out, state_buf(c), c->state_bytes, cudaMemcpyDeviceToHost, c->stream));
  double h = 0.0;
  DG_CUDA(c, cudaMemcpyAsync(&h, &c->sc->t_acc, sizeof h, cudaMemcpyDeviceToHost, c->stream));
  DG_CUDA(c, cudaStreamSynchronize(c->stream));
  if (t_inout_host) *t_inout_host += h;
  return DGRHD_OK;
}

extern "C" int dgrhd_get_counters(dgrhd_ctx* c, int64_t out_host[8], int reset) {
  if (!c || !out_host) return fail(c, DGRHD_EINVAL, "dgrhd_get_counters: NULL argument");
  DevScalars h;
  DG_CUDA(c, cudaMemcpyAsync(&h, c->sc, sizeof h, cudaMemcpyDeviceToHost, c->stream));
  if (reset) {
    DG_CUDA(c, cudaMemsetAsync(c->sc->counters, 0, sizeof h.counters, c->stream));
    DG_CUDA(c, cudaMemsetAsync(&c->sc->n_stages, 0, 2 * sizeof(dg_ull), c->stream));
  }
  DG_CUDA(c, cudaStreamSynchronize(c->stream));
  c->bad_dt_seen = reset ? 0ull : h.n_bad_dt;
  dg_ull sum[5] = {0, 0, 0, 0, 0};
  for (int s = 0; s < DG_NSLOT; ++s)
    for (int k = 0; k < 5; ++k) sum[k] += h.counters[s * DG_SLOT_STRIDE + k];
  out_host[0] = (int64_t)sum[0];
  out_host[1] = (int64_t)sum[1];
  out_host[2] = (int64_t)sum[2];
  out_host[3] = (int64_t)h.n_stages;
  out_host[4] = (int64_t)sum[3];
  out_host[5] = (int64_t)h.n_bad_dt;
  out_host[6] = (int64_t)sum[4];
  out_host[7] = 0;
  return DGRHD_OK;
}

// ------------------------------------------------------------------------------------------------
// context-free batch calls
// ------------------------------------------------------------------------------------------------
static int check_batch(const char* who, int eos, double G, int64_t n, const void* a, const void* b) {
  if (eos != DGRHD_EOS_IDEAL && eos != DGRHD_EOS_TAUB_MATTHEWS)
    return fail(nullptr, DGRHD_EINVAL, "%s: unknown EOS %d", who, eos);
  if (eos == DGRHD_EOS_IDEAL && !(G > 1.0)) return fail(nullptr, DGRHD_EINVAL, "%s: Gamma must be > 1", who);
  if (n < 0 || n > (int64_t)2147483647 * DG_FLAT_NT) return fail(nullptr, DGRHD_EINVAL, "%s: bad n", who);
  if (n > 0 && (!a || !b)) return fail(nullptr, DGRHD_EINVAL, "%s: NULL buffer", who);
  return DGRHD_OK;
}

extern "C" int dgrhd_con2prim_batch(int eos, double gamma_ad, int64_t n, const double* U_dev,
                                    double* W_dev, int* status_dev, void* cuda_stream) {
  int r = check_batch("dgrhd_con2prim_batch", eos, gamma_ad, n, U_dev, W_dev);
  if (r != DGRHD_OK || n == 0) return r;
  const EosPar e = make_eos(eos, gamma_ad);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // two adjacent states per thread with 16-byte accesses when every row is 16-byte aligned
  const bool vec = (n % 2 == 0) && aligned16(U_dev) && aligned16(W_dev);
  const long long nthr = vec ? n / 2 : n;
  const unsigned nb = (unsigned)((nthr + DG_FLAT_NT - 1) / DG_FLAT_NT);
  if (eos == DGRHD_EOS_IDEAL) {
    if (vec) dg_c2p_batch_kernel<0, 2><<<nb, DG_FLAT_NT, 0, st>>>((long long)n, U_dev, W_dev, status_dev, e);
    else dg_c2p_batch_kernel<0, 1><<<nb, DG_FLAT_NT, 0, st>>>((long long)n, U_dev, W_dev, status_dev, e);
  } else {
    if (vec) dg_c2p_batch_kernel<1, 2><<<nb, DG_FLAT_NT, 0, st>>>((long long)n, U_dev, W_dev, status_dev, e);
    else dg_c2p_batch_kernel<1, 1><<<nb, DG_FLAT_NT, 0, st>>>((long long)n, U_dev, W_dev, status_dev, e);
  }
  DG_CUDA(nullptr, cudaGetLastError());
  return DGRHD_OK;
}

extern "C" int dgrhd_con2prim_batch_variant(int eos, int variant, double gamma_ad, int64_t n, const double* U_dev,
                                            double* W_dev, int* status_dev, int max_iter, void* cuda_stream) {
  if (variant == DGRHD_C2P_DEFAULT) return dgrhd_con2prim_batch(eos, gamma_ad, n, U_dev, W_dev, status_dev, cuda_stream);
  if (variant != DGRHD_C2P_ALTERNATE) return fail(nullptr, DGRHD_EINVAL, "dgrhd_con2prim_batch_variant: unknown variant %d", variant);
  int r = check_batch("dgrhd_con2prim_batch_variant", eos, gamma_ad, n, U_dev, W_dev);
  if (r != DGRHD_OK || n == 0) return r;
  if (max_iter < 1) return fail(nullptr, DGRHD_EINVAL, "dgrhd_con2prim_batch_variant: max_iter must be >= 1");
  DG_CUDA(nullptr, dg_launch_c2p_variant(eos, (long long)n, U_dev, W_dev, status_dev, make_eos(eos, gamma_ad), max_iter,
                                         (cudaStream_t)cuda_stream));
  return DGRHD_OK;
}

extern "C" int dgrhd_tm_fallback_count(int64_t* out_host, int reset, void* cuda_stream) {
  if (!out_host) return fail(nullptr, DGRHD_EINVAL, "dgrhd_tm_fallback_count: NULL argument");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  dg_ull h = 0, z = 0;
  DG_CUDA(nullptr, cudaMemcpyFromSymbolAsync(&h, g_tm_fallbacks, sizeof h, 0, cudaMemcpyDeviceToHost, st));
  if (reset) DG_CUDA(nullptr, cudaMemcpyToSymbolAsync(g_tm_fallbacks, &z, sizeof z, 0, cudaMemcpyHostToDevice, st));
  DG_CUDA(nullptr, cudaStreamSynchronize(st));
  *out_host = (int64_t)h;
  return DGRHD_OK;
}

extern "C" int dgrhd_prim2con_batch(int eos, double gamma_ad, int64_t n, const double* W_dev,
                                    double* U_dev, void* cuda_stream) {
  int r = check_batch("dgrhd_prim2con_batch", eos, gamma_ad, n, W_dev, U_dev);
  if (r != DGRHD_OK || n == 0) return r;
  const unsigned nb = (unsigned)((n + DG_FLAT_NT - 1) / DG_FLAT_NT);
  const EosPar e = make_eos(eos, gamma_ad);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (eos == DGRHD_EOS_IDEAL)
    dg_p2c_batch_kernel<0><<<nb, DG_FLAT_NT, 0, st>>>((long long)n, W_dev, U_dev, e);
  else
    dg_p2c_batch_kernel<1><<<nb, DG_FLAT_NT, 0, st>>>((long long)n, W_dev, U_dev, e);
  DG_CUDA(nullptr, cudaGetLastError());
  return DGRHD_OK;
}

// Host-buffer wrapper: chunks of m states go through the staging buffer as [U: 5 x m][W: 5 x m].
extern "C" int dgrhd_con2prim_batch_host(int eos, double gamma_ad, int64_t n, const double* U_host,
                                         double* W_host, void* stage_dev, size_t stage_bytes,
                                         void* cuda_stream) {
  int r = check_batch("dgrhd_con2prim_batch_host", eos, gamma_ad, n, U_host, W_host);
  if (r != DGRHD_OK || n == 0) return r;
  if (!stage_dev || stage_bytes < 160) return fail(nullptr, DGRHD_EINVAL, "dgrhd_con2prim_batch_host: staging buffer too small");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int64_t cap = (int64_t)(stage_bytes / 80) / 2 * 2;      // even chunks keep the rows 16-byte aligned
  double* Ud = (double*)stage_dev;
  for (int64_t s = 0; s < n; s += cap) {
    const int64_t m = (n - s < cap) ? (n - s) : cap;
    double* Wd = Ud + 5 * ((m + 1) / 2 * 2);
    DG_CUDA(nullptr, cudaMemcpy2DAsync(Ud, m * sizeof(double), U_host + s, n * sizeof(double),
                                       m * sizeof(double), 5, cudaMemcpyHostToDevice, st));
    r = dgrhd_con2prim_batch(eos, gamma_ad, m, Ud, Wd, nullptr, cuda_stream);
    if (r != DGRHD_OK) return r;
    DG_CUDA(nullptr, cudaMemcpy2DAsync(W_host + s, n * sizeof(double), Wd, m * sizeof(double),
                                       m * sizeof(double), 5, cudaMemcpyDeviceToHost, st));
  }
  DG_CUDA(nullptr, cudaStreamSynchronize(st));
  return DGRHD_OK;
}

extern "C" int dgrhd_probe_fp64(void* scratch_dev, double* tflops_host, double* sm_mhz_host,
                                void* cuda_stream) {
  if (!scratch_dev || !tflops_host) return fail(nullptr, DGRHD_EINVAL, "dgrhd_probe_fp64: NULL argument");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, nsm = 0, khz = 0;
  DG_CUDA(nullptr, cudaGetDevice(&dev));
  DG_CUDA(nullptr, cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
  DG_CUDA(nullptr, cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
  const int blocks = nsm * 8, iters = 1 << 15;
  cudaEvent_t e0, e1;
  DG_CUDA(nullptr, cudaEventCreate(&e0));
  DG_CUDA(nullptr, cudaEventCreate(&e1));
  double best = 0.0;
  for (int rep = 0; rep < 6; ++rep) {               // the first launches warm the clocks up
    cudaEventRecord(e0, st);
    dg_fp64_probe_kernel<<<blocks, 256, 0, st>>>((double*)scratch_dev, iters, 1.0 + rep);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return cuda_fail(nullptr, e, "dgrhd_probe_fp64"); }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double tf = 2.0 * 8.0 * 256.0 * (double)blocks * (double)iters / (ms * 1e-3) / 1e12;
    if (rep >= 2 && tf > best) best = tf;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *tflops_host = best;
  if (sm_mhz_host) *sm_mhz_host = khz * 1e-3;
  return DGRHD_OK;
}

extern "C" const char* dgrhd_last_error(const dgrhd_ctx* c) { return c ? c->err : g_err; }

// The version string carries the hash of the sources this library was compiled from (build.py passes
// it and reads it back from the file to decide whether a rebuild is due) and says when the kernels are
// the bounds-checked debug ones.
#ifndef DG_SRC_HASH
#define DG_SRC_HASH "unknown"
#endif
#ifdef DG_DEBUG_ASSERTS
#define DG_VERSION_TAIL "+asserts"
#else
#define DG_VERSION_TAIL ""
#endif
extern "C" const char* dgrhd_version(void) { return "dgrhd 0.3 (sm_100a) src=" DG_SRC_HASH DG_VERSION_TAIL; }

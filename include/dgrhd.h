/* dgrhd.h -- C ABI of the B200-native (sm_100a, fp64) hot path of the discontinuous-Galerkin
 * special-relativistic-hydrodynamics method of arxiv 2205.00095 ("PAPER.md"): one SSP
 * Runge-Kutta stage = conserved->primitive recovery at every nodal point, physical flux, element
 * volume integrals, face states + HLL interface flux + surface lift, SSP-RK combine, the
 * physicality-enforcing operator, and the CFL wave-speed reduction.
 *
 * Conventions (all entry points):
 *   - units c = 1; fp64 everywhere; NV = 5 variables.
 *   - conserved  U = [D, Mx, My, Mz, E]                         (PAPER.md:39-43 Eq. 1, :53-56 Eq. 4)
 *     primitive  W = [rho, ux, uy, uz, P], u = gamma*v the spatial 4-velocity
 *   - canonical layout, SoA by variable:  X[v][e][n],  v in 0..4,
 *       e = ix + nx*(iy + ny*iz)  (element),  n = i + N*(j + N*k)  (node in element), N = p+1,
 *       i.e. element of a 5 x ndof array with ndof = nelem_total * N^ndim, row stride ndof.
 *     Nodes are tensor-product Gauss-Lobatto-Legendre points (reading R1).
 *   - every pointer named *_dev is a DEVICE pointer, every pointer named *_host is a HOST pointer.
 *     State pointers handed to dgrhd_rhs / dgrhd_enforce_physicality must be 16-byte aligned (the
 *     kernels move whole nodal lines with 16-byte accesses; EINVAL otherwise); everything else needs
 *     8-byte alignment only (dgrhd_con2prim_batch takes its 16-byte path when it can).  The caller owns all buffers, including the workspace: the library
 *     allocates no device memory and frees none.
 *   - every call returns an int status (DGRHD_OK = 0) and never throws or aborts; argument errors
 *     are detected before any launch.  Numerical trouble is not an error return: it is counted on
 *     the device (see dgrhd_get_counters) or reported per state (dgrhd_con2prim_batch).
 *   - calls enqueue work on the CUDA stream given at create (or in the call) and return without
 *     waiting, except where a *_host out-parameter is documented to synchronise that stream.
 *   - there is no CPU fallback: without a CUDA device every compute call returns DGRHD_ECUDA.
 */
#ifndef DGRHD_H
#define DGRHD_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dgrhd_ctx dgrhd_ctx;          /* opaque, owned by the library, freed by destroy */

enum { DGRHD_EOS_IDEAL = 0,                  /* h = 1 + Gamma/(Gamma-1) Theta   (Eq. 8)  */
       DGRHD_EOS_TAUB_MATTHEWS = 1 };        /* h = 5/2 Theta + 3/2 sqrt(Theta^2+4/9)  (:89 Eq. 10)  */
/* Boundary conditions.  bc[d] = lo + 256*hi (DGRHD_BC_PAIR): lo is the
 * condition at the low end of axis d, hi at the high end; hi = 0 means "the same as lo" (periodic is
 * always both ends), so a plain DGRHD_BC_* value sets both ends. */
enum { DGRHD_BC_PERIODIC = 0,                /* wrap                                                  */
       DGRHD_BC_OUTFLOW = 1,                 /* transmissive: ghost face state = own face state (:621)*/
       DGRHD_BC_REFLECT = 2,                 /* wall: ghost = own state, normal velocity reversed (:541)*/
       DGRHD_BC_DIRICHLET = 3 };             /* ghost = the fixed primitive state bc_state[d][side] (:541)*/
/* (a pair with periodic at exactly one end has no encoding: the macro yields -1, which every call rejects) */
#define DGRHD_BC_PAIR(lo, hi)                                                                      \
  (((hi) == (lo)) ? (lo)                                                                           \
                  : (((lo) == DGRHD_BC_PERIODIC || (hi) == DGRHD_BC_PERIODIC) ? -1 : (lo) + 256 * (hi)))
/* Interface (Riemann) flux: the two-wave HLL flux (reading R9) or the
 * three-wave HLLC flux of Mignone & Bodo (ref [34]); both with lambda_L, lambda_R of Eq. 23-24. */
enum { DGRHD_RIEMANN_HLL = 0, DGRHD_RIEMANN_HLLC = 1 };
/* Shock limiter: none, or the limiter of Moe, Rossmanith & Seal (ref [23]):
 * every cell is rescaled toward its average by theta = min(1, phi((M - wbar)/(w_M - wbar)), phi((m - wbar)/
 * (w_m - wbar))) over the five conserved variables, phi(y) = min(y/1.1, 1), with M, m the extrema of the face
 * neighbours' nodal values widened to wbar +- alpha; or the minmod limiter (ref [24], van Leer) in the same scaling
 * form: theta = min over variables and directions of minmod(a_d, beta D+/2, beta D-/2) / a_d, a_d the cell's linear
 * coefficient along d, D+- the differences of the neighbouring cell averages.  The paper cites both without printing
 * them (readings R18, R19). */
enum { DGRHD_SHOCK_LIMITER_NONE = 0, DGRHD_SHOCK_LIMITER_MOE = 1, DGRHD_SHOCK_LIMITER_MINMOD = 2 };
enum { DGRHD_OK = 0, DGRHD_EINVAL = 1, DGRHD_ENOMEM = 2, DGRHD_ECUDA = 3, DGRHD_ESTATE = 4 };

/* Problem statement: mesh, order, EOS. */
typedef struct {
  int     ndim;            /* 1, 2 or 3                                                            */
  int64_t nelem[3];        /* elements per axis (unused axes must be 1)                            */
  double  xmin[3], xmax[3];/* domain; uniform Cartesian mesh, h_d = (xmax_d - xmin_d)/nelem_d     */
  int     bc[3];           /* DGRHD_BC_* per axis, or DGRHD_BC_PAIR(lo, hi) for different ends             */
  int     order_p;         /* polynomial order 0..4; N = p+1 nodes per direction                  */
  int     eos;             /* DGRHD_EOS_*                                                          */
  double  gamma_ad;        /* adiabatic index Gamma (ideal EOS, > 1); ignored for Taub-Matthews    */
  int     rk_stages;       /* 1 (RK1), 2 (SSPRK2) or 3 (SSPRK3), Shu-Osher form */
  double  eps_q, delta_s;  /* safety knobs of the physicality operator (reading R13c);
                              0,0 = the paper verbatim; defaults used by the tests: 1e-12, 1e-10   */
  int     riemann;         /* DGRHD_RIEMANN_*                                                       */
  int     shock_limiter;   /* DGRHD_SHOCK_LIMITER_*: applied after the physicality operator of every
                              stage of dgrhd_step (two extra small launches per stage)              */
  double  moe_alpha;       /* Moe: tolerance alpha(h) >= 0 (ref [23] suggests ~500 h^1.5); minmod: beta in
                              [1,2] (1 = van Leer's minmod, 2 = generalised slope limiter; 0 means 1)   */
  double  bc_state[3][2][5]; /* Dirichlet ghost primitives [axis][end] = rho, ux, uy, uz, P: all five
                                finite, rho > 0, P > 0 (else the configuration is invalid)            */
} dgrhd_config;

/* Bytes of device workspace dgrhd_create needs for this configuration (0 if cfg is invalid). */
size_t dgrhd_workspace_bytes(const dgrhd_config* cfg);

/* Create a context.  workspace_dev: device buffer of at least dgrhd_workspace_bytes(cfg) bytes,
 * 256-byte aligned, owned by the caller and kept alive until dgrhd_destroy.  cuda_stream: a
 * cudaStream_t (NULL = the legacy default stream) on which every call of this context enqueues.
 * Errors: EINVAL (bad config / NULL / misaligned), ENOMEM (workspace too small), ECUDA. */
int dgrhd_create(const dgrhd_config* cfg, void* workspace_dev, size_t workspace_bytes,
                 void* cuda_stream, dgrhd_ctx** out);
int dgrhd_destroy(dgrhd_ctx* ctx);

/* Options.  DGRHD_OPT_CUDA_GRAPH (default 1): dgrhd_step replays each SSP-RK step (the dt kernel and
 * the fused stage kernels) as one captured CUDA graph instead of 1 + rk_stages launches; results are
 * identical either way. */
enum { DGRHD_OPT_CUDA_GRAPH = 0 };
int dgrhd_set_option(dgrhd_ctx* ctx, int option, int value);

/* Copy the caller's conserved state U_dev[5][ndof] (canonical layout) into / out of the context.
 * set_state also recovers the primitives of every node (Eq. 16) and computes the
 * CFL wave-speed maximum of the new state; it does not apply the physicality operator (R15). */
int dgrhd_set_state(dgrhd_ctx* ctx, const double* U_dev);
int dgrhd_get_state(dgrhd_ctx* ctx, double* U_dev);
/* Primitives W[5][ndof] of the internal state (recovered from it by this call, PAPER.md:128-130
 * Eq. 16: the context keeps only the pressure of its state between stages). */
int dgrhd_get_prims(dgrhd_ctx* ctx, double* W_dev);

/* R = L(U): the DG spatial operator, Eq. 15-18, on caller buffers in the canonical
 * layout: nodal con2prim (Eq. 16), flux (Eq. 2), volume quadrature (Eq. 17), face states and HLL
 * interface flux with lambda_L/R of Eq. 21-24, surface lift (Eq. 18).  Does not touch the internal
 * state.  U_dev and R_dev must not overlap. */
int dgrhd_rhs(dgrhd_ctx* ctx, const double* U_dev, double* R_dev);

/* R = L(U) for callers that cannot allocate device memory: the same operator, kernels and results as
 * dgrhd_rhs (Eq. 15-18), but with no context and no caller workspace.
 *
 * Who this is for.  dgrhd_rhs needs a context, and a context needs a workspace the caller got from
 * cudaMalloc (or from a pool that did).  Some callers have no way to get one at the point where they
 * need the residual: a plug-in inside a host application that has already handed (almost) all of the
 * GPU's memory to its own arena, so that a fresh cudaMalloc fails; a process whose device-memory budget
 * was fixed by its operator up front (an MPS client with a memory limit, a multi-tenant job) and is
 * spent; a latency-critical loop that must not take the device-wide synchronisation and the driver
 * locks that cudaMalloc / cudaFree bring with them.  For them the scratch
 * this operator needs (the pressure of every node, Eq. 16, between its two kernels, plus a few KiB of
 * failure counters) lives in ONE array compiled into the library, a file-scope __device__ array of
 * 12544 + 8 * DGRHD_STATIC_MAX_NDOF bytes (about 8 MiB).  Every GPU on which the library's code is
 * loaded holds that array from load until the process exits, whether or not this call is ever made.
 *
 * The caller still passes the input U_dev[5][ndof] and the output R_dev[5][ndof] (canonical layout, device
 * pointers, 16-byte aligned, not overlapping; the caller's own memory).  cfg describes the mesh as for
 * dgrhd_create (rk_stages, shock_limiter and the physicality knobs are checked but play no part in L).
 * n_c2p_fail_host (or NULL) receives the number of nodes of THIS call whose recovery failed; non-NULL
 * makes the call synchronise cuda_stream, NULL leaves it asynchronous.
 *
 * Limit: ndof = nelem_total * (p+1)^ndim <= DGRHD_STATIC_MAX_NDOF.  A larger mesh is refused with
 * DGRHD_ENOMEM and a message that names both numbers; nothing is launched.  Other errors as dgrhd_rhs
 * (EINVAL for a bad configuration, NULL, misaligned or overlapping pointers; ECUDA).
 *
 * The call itself allocates nothing: no cudaMalloc, cudaFree, stream, event or graph, and no host heap
 * memory.  The first call on each device does a one-time set-up with that device current: it asks the
 * runtime for the device address of the array (the array's name in host code is only a handle, never a
 * pointer a kernel may be given) and opts the stage kernel into its shared-memory size.  Make that first
 * call per device before any stream capture begins; later calls on that device only enqueue a 12 KiB
 * memset of the counters and two kernels.
 *
 * All calls on a device share the one array and it keeps what the previous call left in it.  The call
 * clears the counters itself and overwrites every pressure value before reading it, so calls that run
 * one after another (same stream, or ordered by events) are independent of each other.  Two calls
 * whose kernels can overlap on the GPU (different streams without ordering, or different host threads
 * on different streams) race on the array and both results are undefined: serialise them. */
#define DGRHD_STATIC_MAX_NDOF 1048576
int dgrhd_rhs_static(const dgrhd_config* cfg, const double* U_dev, double* R_dev,
                     int64_t* n_c2p_fail_host, void* cuda_stream);

/* The physicality-enforcing operator of PAPER.md:175-254 (Eq. 25-37), in place on U_dev[5][ndof]
 * (NULL = the internal state, whose primitives are then refreshed): per cell, blend toward the
 * volume average with the largest s in [0,1] that makes every node admissible (D > 0,
 * E > sqrt(D^2+|M|^2)).  flag_dev[n_elem] (or NULL) receives 1 for cells where it acted, 0
 * otherwise; s_dev[n_elem] (or NULL) the blend factor (1 where it did not act, 0 where the cell
 * average itself is inadmissible).  counters_host[2] (or NULL) receives {n_flagged, n_bad_mean} of
 * this call and makes the call synchronise the stream. */
int dgrhd_enforce_physicality(dgrhd_ctx* ctx, double* U_dev, unsigned char* flag_dev,
                              double* s_dev, int64_t counters_host[2]);

/* The shock limiter the context was created with (DGRHD_SHOCK_LIMITER_MOE or _MINMOD), in place on U_dev[5][ndof];
 * theta_dev[n_elem] (or NULL) receives every cell's rescaling factor (1 = untouched).  ESTATE if the
 * context has no shock limiter.  Inside dgrhd_step it runs after the physicality operator of every stage.
 * The stand-alone call touches no counter of dgrhd_get_counters (count theta_dev < 1 instead). */
int dgrhd_shock_limiter(dgrhd_ctx* ctx, double* U_dev, double* theta_dev);

/* CFL time step (formula: DESIGN.md reading R11):
 *   dt = cfl / max_nodes sum_d (2p+1) max(|lambda-_d|, |lambda+_d|) / h_d,  lambda+- of Eq. 21-22.
 * U_dev = NULL uses the internal state.  Synchronises; *dt_host receives dt.  ESTATE if the state has no
 * positive finite wave speed (e.g. con2prim failed everywhere): dt would be infinite. */
int dgrhd_cfl_dt(dgrhd_ctx* ctx, const double* U_dev, double cfl, double* dt_host);

/* Advance the internal state by nsteps SSP-RK steps; each stage is
 *   U <- a U0 + b (U_s + dt L(U_s)), then the physicality operator (R15), then con2prim of the new
 * state; the last stage also reduces the CFL maximum for the next step.
 * dt > 0: fixed step.  dt <= 0: CFL number = -dt, the step is recomputed on the device every step
 * from the state at the start of the step (no host round trip).
 * t_inout_host (or NULL): *t += sum of the steps taken; non-NULL makes the call synchronise.
 * A CFL-mode step that finds no positive finite wave speed in its state (every recovery failed) cannot form
 * dt = CFL / max: it runs with dt = 0 and is counted in n_bad_dt.  Such a state has a non-finite residual, so
 * it comes out non-finite, and every later step is bad too.  With t_inout_host the call reports this as
 * DGRHD_ESTATE (after adding the time actually advanced), once per batch of new bad steps, so that a loop
 * "step until t_end" ends instead of spinning on dt = 0; without it, poll n_bad_dt. */
int dgrhd_step(dgrhd_ctx* ctx, double dt, int nsteps, double* t_inout_host);

/* Device counters accumulated since create / the last reset (synchronises):
 *   out_host[0] n_flagged      cell-activations of the physicality operator inside dgrhd_step
 *   out_host[1] n_bad_mean     cells whose average was itself inadmissible (flattened)
 *   out_host[2] n_c2p_fail     recoveries that failed (inadmissible input or P <= 0), counted in every pass that
 *                              recovers a node: dgrhd_set_state, dgrhd_rhs, the end of every stage and, with a
 *                              shock limiter on, once more for the nodes of every cell it rescaled (so the same
 *                              bad node of the same stage can count twice); 0 means no recovery failed anywhere
 *   out_host[3] n_stages       RK stages executed by dgrhd_step
 *   out_host[4] n_tm_fallback  Taub-Matthews recoveries that took the double-precision closed form
 *                              because the fast route's Newton polish had not converged
 *   out_host[5] n_bad_dt       CFL-mode steps whose wave-speed maximum was not a positive finite
 *                              number: they ran with dt = 0 instead of dt = inf (see dgrhd_step)
 *   out_host[6] n_shock_limited  cell-rescalings (theta < 1) by the shock limiter; out_host[7] reserved (0)
 * reset != 0 zeroes them afterwards. */
int dgrhd_get_counters(dgrhd_ctx* ctx, int64_t out_host[8], int reset);

/* Conserved -> primitive recovery of a flat SoA batch U_dev[5][n] -> W_dev[5][n]:
 * ideal EOS by Newton iteration on the quartic of Eq. 59 (beta = 2w/(1+w^2), Eq. 58; small-xi
 * series Eq. 60; finishing Eq. 55-57); Taub-Matthews by the analytic cubic Eq. 61-75.
 * status_dev[n] (or NULL): 0 ok; 1 input not admissible by Eq. 25 (outputs NaN); 2 recovered
 * pressure not positive / non-finite.  Enqueues on cuda_stream; does not synchronise.  n = 0 ok. */
int dgrhd_con2prim_batch(int eos, double gamma_ad, int64_t n, const double* U_dev, double* W_dev,
                         int* status_dev, void* cuda_stream);

/* The paper's comparison variants of the recovery ("four algorithms in all", the study of
 * section 3.3, :405-449), same layout and status codes as dgrhd_con2prim_batch:
 *   DGRHD_C2P_DEFAULT    the hot-path solvers (ideal: Newton on Eq. 59; Taub-Matthews: analytic cubic)
 *   DGRHD_C2P_ALTERNATE  ideal EOS by the analytic quartic in beta (Eq. 39-57, after Ryu et al.);
 *                        Taub-Matthews by Brent's method on Eq. 61, bracket gamma in [1,200] expanded
 *                        if needed, at most max_iter iterations (>= 1; the paper's Fig. 2 uses 25, 50) */
enum { DGRHD_C2P_DEFAULT = 0, DGRHD_C2P_ALTERNATE = 1 };
int dgrhd_con2prim_batch_variant(int eos, int variant, double gamma_ad, int64_t n, const double* U_dev,
                                 double* W_dev, int* status_dev, int max_iter, void* cuda_stream);

/* Number of Taub-Matthews recoveries of the context-free batch calls (all streams of the current
 * device) that took the double-precision fallback since the last reset (see n_tm_fallback above).
 * Synchronises cuda_stream. */
int dgrhd_tm_fallback_count(int64_t* out_host, int reset, void* cuda_stream);

/* Primitive -> conserved, Eq. 4, flat SoA batch W_dev[5][n] -> U_dev[5][n]. */
int dgrhd_prim2con_batch(int eos, double gamma_ad, int64_t n, const double* W_dev, double* U_dev,
                         void* cuda_stream);

/* Host-buffer convenience wrapper around dgrhd_con2prim_batch: copies U_host[5][n] to the device
 * (chunked, through the caller's 16-byte aligned staging buffer stage_dev of stage_bytes >= 80 bytes
 * per state of one chunk, at least 160), runs the kernel, copies W_host[5][n] back, synchronises.  Used for end-to-end timing. */
int dgrhd_con2prim_batch_host(int eos, double gamma_ad, int64_t n, const double* U_host,
                              double* W_host, void* stage_dev, size_t stage_bytes,
                              void* cuda_stream);

/* End-to-end wrapper with HOST buffers (pinned memory for full copy speed): copies
 * U_host_in[5][ndof] to the device, dgrhd_set_state, dgrhd_step(dt, nsteps), copies the new state
 * to U_host_out[5][ndof], synchronises.  *t_inout_host (or NULL) += elapsed time. */
int dgrhd_run_host(dgrhd_ctx* ctx, const double* U_host_in, double* U_host_out, double dt,
                   int nsteps, double* t_inout_host);

/* Measurement aid: sustained FP64 FMA throughput of the current device in TFLOP/s (best of four
 * ~2 ms launches of a register-only DFMA kernel, timed with CUDA events on cuda_stream; synchronises).
 * It is the measured denominator of the "alu" roofline bench.py reports.  scratch_dev: >= 8 bytes of
 * device memory.  sm_mhz_host (or NULL) receives the device's nominal maximum SM clock. */
int dgrhd_probe_fp64(void* scratch_dev, double* tflops_host, double* sm_mhz_host, void* cuda_stream);

/* Text of the last error of this context (ctx = NULL: of the last context-free call on this
 * thread).  Never NULL; valid until the next call on the same context / thread. */
const char* dgrhd_last_error(const dgrhd_ctx* ctx);

/* Library version string: "dgrhd 0.3 (sm_100a) src=<16 hex digits>", the hash being that of the sources the
 * library was compiled from (paper_2205_00095_b200/build.py); the bounds-checked debug build appends "+asserts". */
const char* dgrhd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DGRHD_H */

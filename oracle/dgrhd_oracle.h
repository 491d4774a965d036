/* dgrhd_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU restatement of the DG special-relativistic-hydro stage of
 * arxiv 2205.00095 ("PAPER.md"), written from the paper's equations in the paper's order.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may use anything under oracle/.  It shares no code, header, table or constant generator
 * with paper_2205_00095_b200/ (the CUDA path); neither includes the other.
 *
 * Units: c = 1 throughout (PAPER.md keeps c; every workload here is in units of c).
 * Layout (canonical, SoA by variable): X[v][e][n], v in {D|rho, Mx|ux, My|uy, Mz|uz, E|P},
 *   e = ix + nx*(iy + ny*iz), n = i + N*(j + N*k), N = p+1.   Primitive velocity is the
 *   spatial 4-velocity u = gamma*v.
 *
 * Readings of the paper (R#) are the ones listed in DESIGN.md "Readings".
 */
#ifndef DGRHD_ORACLE_H
#define DGRHD_ORACLE_H
#include <stdint.h>

enum { ORC_EOS_IDEAL = 0, ORC_EOS_TM = 1 };
/* Boundary conditions.  bc[d] = lo + 256*hi: lo = condition at the low
 * end of axis d, hi = at the high end (hi = 0: the same as lo -- periodic is always both ends).
 *   OUTFLOW    ghost face state = own face state (reading R12)
 *   REFLECT    ghost = own state with the normal velocity reversed (a wall, :541 test 5)
 *   DIRICHLET  ghost = the fixed primitive state bc_state[d][side] (:541 tests 1-4) */
enum { ORC_BC_PERIODIC = 0, ORC_BC_OUTFLOW = 1, ORC_BC_REFLECT = 2, ORC_BC_DIRICHLET = 3 };
enum { ORC_RIEMANN_HLL = 0, ORC_RIEMANN_HLLC = 1 };

typedef struct {
  int     ndim;          /* 1,2,3 */
  int64_t nelem[3];      /* elements per axis (unused = 1) */
  double  xmin[3], xmax[3];
  int     bc[3];
  int     order_p;       /* 0..4 */
  int     eos;
  double  gamma_ad;
  int     rk_stages;     /* 1,2,3 */
  double  eps_q, delta_s;
  int     riemann;       /* ORC_RIEMANN_*: interface flux */
  int     shock_limiter; /* 0 none; 1 the limiter of Moe, Rossmanith & Seal (PAPER.md:126, :551 ref [23]);
                            2 the minmod limiter (PAPER.md:126, :597 ref [24]); applied after the
                            physicality operator of every stage.  PARITY UNPINNED: the paper cites both
                            without printing them (readings R18, R19) */
  double  moe_alpha;     /* Moe: tolerance alpha(h) >= 0 (ref [23] suggests ~ 500 h^1.5), absolute;
                            minmod: beta in [1,2] (0 = 1) */
  double  bc_state[3][2][5];   /* Dirichlet ghost primitives [axis][side] = rho, ux, uy, uz, P */
} orc_config;

/* O4: GLL tables for N = p+1 nodes: x[N], w[N], D[q*N+i] = l_i'(x_q). */
void orc_gll(int N, double *x, double *w, double *D);

/* O1 */
double orc_enthalpy(int eos, double G, double rho, double P);
double orc_cs2(int eos, double G, double rho, double P);
void   orc_prim2con(int eos, double G, const double W[5], double U[5]);
void   orc_flux(int eos, double G, const double W[5], int dir, double F[5]);
void   orc_wavespeeds(int eos, double G, const double W[5], int dir, double *lm, double *lp);
void   orc_hll(int eos, double G, const double WL[5], const double WR[5], int dir, double F[5]);
/* HLLC of Mignone & Bodo (PAPER.md:161 ref [34]); lstar_out (may be NULL) receives lambda*;
 * UsL/UsR (may be NULL) the two star states */
void   orc_hllc(int eos, double G, const double WL[5], const double WR[5], int dir, double F[5],
                double *lstar_out, double UsL[5], double UsR[5]);

/* O2/O3: returns status 0 ok, 1 inadmissible input (W = NaN), 2 solver/pressure failure.
 * niter_out (may be NULL) receives the Newton iteration count (ideal EOS). */
int    orc_con2prim(int eos, double G, const double U[5], double W[5], int *niter_out);
/* ideal EOS Newton with a caller-fixed iteration count and no stopping test (Fig. 2 protocol) */
int    orc_con2prim_ideal_fixed(double G, const double U[5], double W[5], int niter);

/* the paper's comparison variants (section 3.3): variant 0 = orc_con2prim; 1 = ideal EOS by the analytic
 * quartic (Eq. 39-57) / Taub-Matthews by Brent's method on Eq. 61 with at most max_iter iterations */
int    orc_con2prim_variant(int eos, int variant, double G, const double U[5], double W[5], int max_iter,
                            int *niter_out);
void   orc_con2prim_variant_batch(int eos, int variant, double G, int64_t n, const double *U, double *W,
                                  int *status, int max_iter);

void   orc_prim2con_batch(int eos, double G, int64_t n, const double *W, double *U);
void   orc_con2prim_batch(int eos, double G, int64_t n, const double *U, double *W, int *status);

/* O7 building blocks (exposed for the pins) */
int    orc_admissible(const double U[5], double eps);
double orc_limiter_node_s(const double Ubar[5], const double Ui[5], double eps_q);

/* O5..O7, R10, R11 on the canonical layout; ndof = nelem_total * N^ndim */
int64_t orc_ndof(const orc_config *c);
void   orc_rhs(const orc_config *c, const double *U, double *R, int64_t *n_c2p_fail);
void   orc_enforce_physicality(const orc_config *c, double *U, unsigned char *flag, double *s,
                               int64_t counters[2]);
/* The shock limiter of Moe et al. (reading R18), in place; theta[n_e] (may be NULL) receives the
 * rescaling factor of every cell; returns the number of cells with theta < 1. */
int64_t orc_shock_limiter(const orc_config *c, double *U, double *theta);
double orc_cfl_dt(const orc_config *c, const double *U, double cfl);
/* dt > 0 fixed; dt <= 0: CFL number -dt, recomputed every step.  counters[3] accumulates
 * n_flagged, n_bad_mean, n_c2p_fail over all stages. */
void   orc_step(const orc_config *c, double *U, double dt, int nsteps, double *t_inout,
                int64_t counters[3]);
int    orc_num_threads(void);
#endif

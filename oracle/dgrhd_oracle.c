/* dgrhd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see dgrhd_oracle.h).
 *
 * Plain fp64 CPU oracle for one SSP-RK stage of the DG-RHD method of arxiv 2205.00095.
 * Every function cites the PAPER.md passage it restates.  Build: gcc -O2 -ffp-contract=off
 * (no fast-math, no FMA contraction) [-fopenmp: outer loops over elements / states only, which
 * does not change any arithmetic or summation order].
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): every function the paper prints is pinned; see DESIGN.md
 * "Oracle pins".  PARITY UNPINNED BY THE PAPER: orc_shock_limiter (the Moe limiter and the minmod limiter),
 * which the paper cites (refs [23], [24]) without printing; they are restated in DESIGN.md readings R18 / R19.
 * What is pinned is the reading: the Moe branch by hand-worked cases (tests/golden/moe_limiter_cases.txt) and
 * its properties, the minmod branch by its reduction to van Leer's minmod and its properties.
 */
#include "dgrhd_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------------
 * O4  Basis: Gauss-Lobatto-Legendre nodes/weights, N = p+1 (reading R1; PAPER.md:110-119 gives a
 * nodal Lagrange basis, Eq. 13-14, without naming the node family).  D[q*N+i] = l_i'(x_q).
 * ------------------------------------------------------------------------------------------ */
void orc_gll(int N, double *x, double *w, double *D) {
  switch (N) {
    case 1: x[0] = 0.0; w[0] = 2.0; break;
    case 2: x[0] = -1.0; x[1] = 1.0; w[0] = 1.0; w[1] = 1.0; break;
    case 3: x[0] = -1.0; x[1] = 0.0; x[2] = 1.0;
            w[0] = 1.0 / 3.0; w[1] = 4.0 / 3.0; w[2] = 1.0 / 3.0; break;
    case 4: x[0] = -1.0; x[1] = -sqrt(1.0 / 5.0); x[2] = sqrt(1.0 / 5.0); x[3] = 1.0;
            w[0] = 1.0 / 6.0; w[1] = 5.0 / 6.0; w[2] = 5.0 / 6.0; w[3] = 1.0 / 6.0; break;
    case 5: x[0] = -1.0; x[1] = -sqrt(3.0 / 7.0); x[2] = 0.0; x[3] = sqrt(3.0 / 7.0); x[4] = 1.0;
            w[0] = 1.0 / 10.0; w[1] = 49.0 / 90.0; w[2] = 32.0 / 45.0; w[3] = 49.0 / 90.0;
            w[4] = 1.0 / 10.0; break;
    default: return;
  }
  /* l_i'(x_q) = sum_{m!=i} 1/(x_i-x_m) prod_{k!=i,m} (x_q-x_k)/(x_i-x_k)   (Lagrange, Eq. 14) */
  for (int q = 0; q < N; ++q)
    for (int i = 0; i < N; ++i) {
      double s = 0.0;
      for (int m = 0; m < N; ++m) {
        if (m == i) continue;
        double t = 1.0 / (x[i] - x[m]);
        for (int k = 0; k < N; ++k) {
          if (k == i || k == m) continue;
          t *= (x[q] - x[k]) / (x[i] - x[k]);
        }
        s += t;
      }
      D[q * N + i] = s;
    }
}

/* ------------------------------------------------------------------------------------------
 * O1  EOS, prim->con, flux, wave speeds  (PAPER.md:45-56 Eq. 2-4, :79-93 Eq. 8-11, :163-167)
 * ------------------------------------------------------------------------------------------ */
/* Eq. 8 (ideal) / Eq. 10 (Taub-Matthews), Theta = P/rho, c = 1 */
double orc_enthalpy(int eos, double G, double rho, double P) {
  double Th = P / rho;
  if (eos == ORC_EOS_IDEAL) return 1.0 + G / (G - 1.0) * Th;
  return 2.5 * Th + 1.5 * sqrt(Th * Th + 4.0 / 9.0);
}

/* Eq. 9 (ideal) / Eq. 11 (Taub-Matthews) */
double orc_cs2(int eos, double G, double rho, double P) {
  double Th = P / rho;
  if (eos == ORC_EOS_IDEAL) return G * Th / orc_enthalpy(eos, G, rho, P);
  double r = sqrt(Th * Th + 4.0 / 9.0);
  return (3.0 * Th * Th + 5.0 * Th * r) / (12.0 * Th * Th + 2.0 + 12.0 * Th * r);
}

/* Eq. 4 with W = [rho, u, P], u = gamma v, gamma = sqrt(1+|u|^2) */
void orc_prim2con(int eos, double G, const double W[5], double U[5]) {
  double rho = W[0], P = W[4];
  double u2 = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
  double g = sqrt(1.0 + u2);
  double h = orc_enthalpy(eos, G, rho, P);
  U[0] = g * rho;                 /* D = gamma rho          */
  U[1] = g * rho * h * W[1];      /* M = gamma rho h u      */
  U[2] = g * rho * h * W[2];
  U[3] = g * rho * h * W[3];
  U[4] = g * g * rho * h - P;     /* E = gamma^2 rho h - P  */
}

/* Eq. 2 in direction dir:  [rho u_d, rho h u u_d + P e_d, gamma rho h u_d]
 *   = [D v_d, M v_d + P e_d, (E+P) v_d]  with v = u/gamma */
void orc_flux(int eos, double G, const double W[5], int dir, double F[5]) {
  double U[5];
  orc_prim2con(eos, G, W, U);
  double u2 = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
  double g = sqrt(1.0 + u2);
  double vd = W[1 + dir] / g;
  F[0] = U[0] * vd;
  F[1] = U[1] * vd;
  F[2] = U[2] * vd;
  F[3] = U[3] * vd;
  F[1 + dir] += W[4];
  F[4] = (U[4] + W[4]) * vd;
}

/* Eq. 21-22, "v_x" = velocity component normal to the face */
void orc_wavespeeds(int eos, double G, const double W[5], int dir, double *lm, double *lp) {
  double u2 = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
  double g2 = 1.0 + u2;
  double vd = W[1 + dir] / sqrt(g2);
  double cs2 = orc_cs2(eos, G, W[0], W[4]);
  double sig = cs2 / (g2 * (1.0 - cs2));                       /* Eq. 22 */
  double root = sqrt(sig * (1.0 - vd * vd + sig));
  *lm = (vd - root) / (1.0 + sig);                             /* Eq. 21 */
  *lp = (vd + root) / (1.0 + sig);
}

/* HLL two-wave flux (PAPER.md:161 cites Schneider et al.; formula not printed: reading R9),
 * lambda_L, lambda_R by Eq. 23-24; U_{L,R} recomputed from W_{L,R} by Eq. 4 (reading R8). */
void orc_hll(int eos, double G, const double WL[5], const double WR[5], int dir, double F[5]) {
  double lmL, lpL, lmR, lpR;
  orc_wavespeeds(eos, G, WL, dir, &lmL, &lpL);
  orc_wavespeeds(eos, G, WR, dir, &lmR, &lpR);
  double lL = fmin(lmL, lmR);                                   /* Eq. 23 */
  double lR = fmax(lpL, lpR);                                   /* Eq. 24 */
  double FL[5], FR[5], UL[5], UR[5];
  orc_flux(eos, G, WL, dir, FL);
  orc_flux(eos, G, WR, dir, FR);
  if (lL >= 0.0) { for (int v = 0; v < 5; ++v) F[v] = FL[v]; return; }
  if (lR <= 0.0) { for (int v = 0; v < 5; ++v) F[v] = FR[v]; return; }
  orc_prim2con(eos, G, WL, UL);
  orc_prim2con(eos, G, WR, UR);
  for (int v = 0; v < 5; ++v)
    F[v] = (lR * FL[v] - lL * FR[v] + lL * lR * (UR[v] - UL[v])) / (lR - lL);
}

/* HLLC three-wave flux.  PAPER.md:126/:161/:551 names it ("HLL and HLLC variants ... Mignone and
 * Bodo [34]") without printing it; this is ref [34]'s construction, with lambda_L, lambda_R of
 * Eq. 23-24 as for HLL.  From the HLL state and flux
 *   U^hll = (lR U_R - lL U_L + F_L - F_R)/(lR - lL),  F^hll = (lR F_L - lL F_R + lL lR (U_R - U_L))/(lR - lL)
 * the contact speed lambda* is the root with the minus sign of
 *   F_E^hll l^2 - (E^hll + F_m^hll) l + m^hll = 0        (m = momentum normal to the face),
 * p* = -F_E^hll l* + F_m^hll, and for K = L, R (v, p: normal velocity and pressure of side K):
 *   D*  = D (lK - v)/(lK - l*),            m_t* = m_t (lK - v)/(lK - l*)   (transverse momenta),
 *   m*  = (m (lK - v) + p* - p)/(lK - l*), E*   = (E (lK - v) + p* l* - p v)/(lK - l*);
 * flux:  F_L (lL >= 0);  F_L + lL (U*_L - U_L) (lL < 0 <= l*);  F_R + lR (U*_R - U_R) (l* < 0 <= lR);
 * F_R (lR < 0).  A vanishing leading coefficient (|F_E^hll| tiny) makes the quadratic linear. */
void orc_hllc(int eos, double G, const double WL[5], const double WR[5], int dir, double F[5],
              double *lstar_out, double UsL_out[5], double UsR_out[5]) {
  double lmL, lpL, lmR, lpR;
  orc_wavespeeds(eos, G, WL, dir, &lmL, &lpL);
  orc_wavespeeds(eos, G, WR, dir, &lmR, &lpR);
  double lL = fmin(lmL, lmR);                                   /* Eq. 23 */
  double lR = fmax(lpL, lpR);                                   /* Eq. 24 */
  double FL[5], FR[5], UL[5], UR[5], Uh[5], Fh[5];
  orc_flux(eos, G, WL, dir, FL);
  orc_flux(eos, G, WR, dir, FR);
  orc_prim2con(eos, G, WL, UL);
  orc_prim2con(eos, G, WR, UR);
  for (int v = 0; v < 5; ++v) {
    Uh[v] = (lR * UR[v] - lL * UL[v] + FL[v] - FR[v]) / (lR - lL);
    Fh[v] = (lR * FL[v] - lL * FR[v] + lL * lR * (UR[v] - UL[v])) / (lR - lL);
  }
  const int im = 1 + dir;
  double a = Fh[4], b = -(Uh[4] + Fh[im]), cc = Uh[im];
  double ls;
  if (fabs(a) > 1e-14 * fabs(b)) {
    double disc = sqrt(fmax(b * b - 4.0 * a * cc, 0.0));
    /* the root with the minus sign, written without cancellation (b < 0): 2c / (-b + disc) */
    ls = 2.0 * cc / (-b + disc);
  } else {
    ls = -cc / b;
  }
  double ps = -Fh[4] * ls + Fh[im];
  double Us[2][5];
  for (int K = 0; K < 2; ++K) {
    const double *U = K ? UR : UL, *W = K ? WR : WL;
    double lK = K ? lR : lL;
    double g = sqrt(1.0 + W[1] * W[1] + W[2] * W[2] + W[3] * W[3]);
    double v = W[im] / g, p = W[4];
    double den = lK - ls;
    for (int k = 0; k < 4; ++k) Us[K][k] = U[k] * (lK - v) / den;
    Us[K][im] = (U[im] * (lK - v) + ps - p) / den;
    Us[K][4] = (U[4] * (lK - v) + ps * ls - p * v) / den;
  }
  if (lstar_out) *lstar_out = ls;
  if (UsL_out) for (int v = 0; v < 5; ++v) UsL_out[v] = Us[0][v];
  if (UsR_out) for (int v = 0; v < 5; ++v) UsR_out[v] = Us[1][v];
  if (lL >= 0.0) { for (int v = 0; v < 5; ++v) F[v] = FL[v]; return; }
  if (lR <= 0.0) { for (int v = 0; v < 5; ++v) F[v] = FR[v]; return; }
  if (ls >= 0.0) { for (int v = 0; v < 5; ++v) F[v] = FL[v] + lL * (Us[0][v] - UL[v]); }
  else           { for (int v = 0; v < 5; ++v) F[v] = FR[v] + lR * (Us[1][v] - UR[v]); }
}

/* ------------------------------------------------------------------------------------------
 * O7 predicate: Eq. 25 with the PLUS sign under the root (reading R13a; Eq. 27/31/32), the
 * safety factor (1-eps) on E (R13c), separately rounded operations in this order (R13e).
 * NaN anywhere => not admissible.
 * ------------------------------------------------------------------------------------------ */
int orc_admissible(const double U[5], double eps) {
  double D = U[0];
  double m2 = D * D;
  m2 = m2 + U[1] * U[1];
  m2 = m2 + U[2] * U[2];
  m2 = m2 + U[3] * U[3];
  double Es = (1.0 - eps) * U[4];
  return (D > 0.0) && (Es > sqrt(m2));
}

/* ------------------------------------------------------------------------------------------
 * O2  con2prim, ideal EOS: Newton on the quartic of Eq. 59 in w, beta = 2w/(1+w^2) (Eq. 58,
 * reading R5), finishing by Eq. 55-57.  PAPER.md:262-263 (Eq. 38), :329-345.
 * ------------------------------------------------------------------------------------------ */
static void ideal_coeffs(double al, double xi, double eta, double c[5]) {
  c[4] = (al - 1.0) * xi;            /* Eq. 59, w^4 */
  c[3] = -2.0 * (al * eta + 1.0);    /* w^3 */
  c[2] = 2.0 * (al + 1.0) * xi;      /* w^2 */
  c[1] = -2.0 * (al * eta - 1.0);    /* w^1 */
  c[0] = (al - 1.0) * xi;            /* w^0 */
}

static void ideal_finish(double G, const double U[5], double Mabs, double w, double W[5]) {
  double D = U[0], E = U[4];
  double w2 = w * w;
  double beta = 2.0 * w / (1.0 + w2);                 /* Eq. 58 */
  double ig = (1.0 - w2) / (1.0 + w2);                /* 1/gamma = sqrt(1-beta^2), exact identity */
  double rho = D * ig;                                /* Eq. 55 */
  double nx = 0.0, ny = 0.0, nz = 0.0;
  if (Mabs > 0.0) { nx = U[1] / Mabs; ny = U[2] / Mabs; nz = U[3] / Mabs; }
  double ug = 2.0 * w / (1.0 - w2);                   /* gamma*beta */
  W[0] = rho;
  W[1] = ug * nx;                                     /* u = gamma v, v = beta M/|M|  (Eq. 56) */
  W[2] = ug * ny;
  W[3] = ug * nz;
  W[4] = (G - 1.0) * (E - beta * Mabs - rho);         /* Eq. 57, M.v = beta |M| */
}

static int finite5(const double W[5]) {
  for (int v = 0; v < 5; ++v) if (!isfinite(W[v])) return 0;
  return 1;
}

static int con2prim_ideal(double G, const double U[5], double W[5], int *niter_out, int fixed_iter) {
  double D = U[0], E = U[4];
  double Mabs = sqrt(U[1] * U[1] + U[2] * U[2] + U[3] * U[3]);
  double xi = Mabs / D, eta = E / D;                  /* Eq. 38 */
  double al = G / (G - 1.0);
  double w;
  int it = 0;
  if (xi == 0.0) {
    w = 0.0;
  } else if (xi < 1e-4 && fixed_iter < 0) {
    /* Eq. 60, small-xi cubic series (reading R4) */
    double a1 = al * eta - 1.0;
    double a14 = a1 * a1 * a1 * a1;
    w = (al - 1.0) / (2.0 * a1) * xi +
        (al - 1.0) * (al - 1.0) / (8.0 * a14) * ((al + 3.0) * (al * eta + 1.0) - 4.0 * (al + 1.0)) *
            xi * xi * xi;
  } else {
    double c[5];
    ideal_coeffs(al, xi, eta, c);
    double b0 = xi / eta;                             /* reading R2: beta_0 = |M|/E >= beta */
    w = b0 / (1.0 + sqrt(1.0 - b0 * b0));
    int maxit = fixed_iter >= 0 ? fixed_iter : 16;    /* reading R3 */
    for (it = 0; it < maxit;) {
      double p = (((c[4] * w + c[3]) * w + c[2]) * w + c[1]) * w + c[0];
      double dp = ((4.0 * c[4] * w + 3.0 * c[3]) * w + 2.0 * c[2]) * w + c[1];
      double dw = p / dp;
      w = w - dw;
      ++it;
      if (fixed_iter < 0 && fabs(dw) <= 1e-14 * w) break;
    }
  }
  if (niter_out) *niter_out = it;
  ideal_finish(G, U, Mabs, w, W);
  if (!(w >= 0.0 && w < 1.0) || !finite5(W) || !(W[4] > 0.0)) return 2;
  return 0;
}

/* ------------------------------------------------------------------------------------------
 * O3  con2prim, Taub-Matthews: analytic cubic in W = gamma^2 - 1, Eq. 61-73, finishing by
 * Eq. 74-75, safeguards of reading R7.
 * ------------------------------------------------------------------------------------------ */
static int con2prim_tm(const double U[5], double Wp[5]) {
  double D = U[0], E = U[4];
  double Mabs = sqrt(U[1] * U[1] + U[2] * U[2] + U[3] * U[3]);
  double xi = Mabs / D, eta = E / D;                  /* Eq. 38 */
  double x2 = xi * xi, e2 = eta * eta;
  double dif = (eta - xi) * (eta + xi);               /* eta^2 - xi^2 (R7) */
  double den = dif * dif;
  double sum = e2 + x2;
  double br = 4.0 * sum - (x2 + 1.0);
  double c1 = (sum * br - 14.0 * x2 * e2) / (2.0 * den);      /* Eq. 62 */
  double c2 = (br * br - 57.0 * x2 * e2) / (16.0 * den);      /* Eq. 63 */
  double c3 = -9.0 * x2 * e2 / (16.0 * den);                  /* Eq. 64 */
  double Q = (3.0 * c2 - c1 * c1) / 9.0;                      /* Eq. 66 */
  double R = (9.0 * c1 * c2 - 27.0 * c3 - 2.0 * c1 * c1 * c1) / 54.0;   /* Eq. 67 */
  double d = Q * Q * Q + R * R;                               /* Eq. 65 */
  double Wv;
  if (d < 0.0) {
    double arg = R / sqrt(-(Q * Q * Q));
    if (arg > 1.0) arg = 1.0;
    if (arg < -1.0) arg = -1.0;
    double iota = acos(arg);                                  /* Eq. 70 */
    Wv = 2.0 * sqrt(-Q) * cos(iota / 3.0) - c1 / 3.0;         /* Eq. 69 */
  } else {
    double sd = sqrt(d);
    Wv = -c1 / 3.0 + cbrt(R + sd) + cbrt(R - sd);             /* Eq. 71-73, real cube roots */
  }
  if (Wv < 0.0) Wv = 0.0;                                     /* R7 */
  /* R7b: one Newton correction of the root on the cubic of Eq. 61 itself.  The closed forms above
   * return W as a difference of O(c1) terms, i.e. with an ABSOLUTE error ~1e-16 c1, which is a
   * large relative error when W = gamma^2-1 -> 0; f(W) = ((W+c1)W+c2)W+c3 has no such cancellation
   * near the (simple, only positive) root, so one step restores full relative accuracy. */
  {
    double f = ((Wv + c1) * Wv + c2) * Wv + c3;
    double df = (3.0 * Wv + 2.0 * c1) * Wv + c2;
    double Wn = Wv - f / df;
    if (isfinite(Wn)) Wv = Wn;
    if (Wv < 0.0) Wv = 0.0;
  }
  double g = sqrt(Wv + 1.0);                                  /* Eq. 74 */
  double beta = sqrt(Wv / (Wv + 1.0));
  double rho = D / g;
  double nx = 0.0, ny = 0.0, nz = 0.0;
  if (Mabs > 0.0) { nx = U[1] / Mabs; ny = U[2] / Mabs; nz = U[3] / Mabs; }
  double ug = sqrt(Wv);                                       /* gamma beta */
  double X = E - beta * Mabs;                                 /* E - M.v */
  Wp[0] = rho;
  Wp[1] = ug * nx;
  Wp[2] = ug * ny;
  Wp[3] = ug * nz;
  Wp[4] = (X - rho) * (X + rho) / (3.0 * X);                  /* Eq. 75 */
  if (!finite5(Wp) || !(Wp[4] > 0.0)) return 2;
  return 0;
}

/* ------------------------------------------------------------------------------------------
 * The paper's two comparison variants of con2prim ("four algorithms in all"; the
 * section 3.3 study, :405-449).  SURVEY.md 8(f).3.
 *
 * (1) Ideal EOS, ANALYTIC route (:269-323, Eq. 39-57, after Ryu et al. [15]): the physical root of
 *   beta^4 + a3 beta^3 + a2 beta^2 + a1 beta + a0 = 0     (Eq. 39; the beta^3 term is missing in the
 *   extracted text -- with it the true beta is a root to 1e-50, reading R17)
 * with a0..a3 of Eq. 40-43, by Ferrari's factorisation: x = real root of the resolvent cubic
 * x^3 + i1 x^2 + i2 x + i3 (Eq. 51-53; Eq. 48 reads 9 i1 i2, Eq. 49 uses i1^2 = a2^2), trigonometric
 * form for T < 0 -- 2 sqrt(-S) cos(acos(R / sqrt(-S^3)) / 3) - i1/3, which is what the garbled
 * Eq. 47 encodes ((R^2 - T)^(1/6) = sqrt(-S)) -- else Cardano; B, C of Eq. 45-46; beta by Eq. 44;
 * finishing Eq. 55-57.
 * ------------------------------------------------------------------------------------------ */
static int con2prim_ideal_analytic(double G, const double U[5], double W[5]) {
  double D = U[0], E = U[4];
  double Mabs = sqrt(U[1] * U[1] + U[2] * U[2] + U[3] * U[3]);
  double xi = Mabs / D, eta = E / D;                                   /* Eq. 38 */
  double beta;
  if (xi == 0.0) {
    beta = 0.0;
  } else {
    double g1 = G - 1.0, den = g1 * g1 * (xi * xi + 1.0);
    double a3 = -2.0 * G * g1 * xi * eta / den;                        /* Eq. 40 */
    double a2 = (G * G * eta * eta + 2.0 * g1 * xi * xi - g1 * g1) / den;   /* Eq. 41 */
    double a1 = -2.0 * G * xi * eta / den;                             /* Eq. 42 */
    double a0 = xi * xi / den;                                         /* Eq. 43 */
    double i1 = -a2;                                                   /* Eq. 51 */
    double i2 = a3 * a1 - 4.0 * a0;                                    /* Eq. 52 */
    double i3 = 4.0 * a2 * a0 - a1 * a1 - a3 * a3 * a0;                /* Eq. 53 */
    double R = (9.0 * i1 * i2 - 27.0 * i3 - 2.0 * i1 * i1 * i1) / 54.0;   /* Eq. 48 */
    double S = (3.0 * i2 - i1 * i1) / 9.0;                             /* Eq. 49 */
    double T = R * R + S * S * S;                                      /* Eq. 50 */
    double x;
    if (T < 0.0) {                                                     /* Eq. 47 */
      double arg = R / sqrt(-(S * S * S));
      if (arg > 1.0) arg = 1.0;
      if (arg < -1.0) arg = -1.0;
      x = 2.0 * sqrt(-S) * cos(acos(arg) / 3.0) - i1 / 3.0;
    } else {
      double sT = sqrt(T);
      x = cbrt(R + sT) + cbrt(R - sT) - i1 / 3.0;
    }
    double B = 0.5 * (a3 + sqrt(a3 * a3 - 4.0 * a2 + 4.0 * x));        /* Eq. 45 */
    double C = 0.5 * (x - sqrt(x * x - 4.0 * a0));                     /* Eq. 46 */
    beta = 0.5 * (-B + sqrt(B * B - 4.0 * C));                         /* Eq. 44 */
  }
  double rho = D * sqrt(1.0 - beta * beta);                            /* Eq. 55 */
  double g = 1.0 / sqrt(1.0 - beta * beta);
  double nx = 0.0, ny = 0.0, nz = 0.0;
  if (Mabs > 0.0) { nx = U[1] / Mabs; ny = U[2] / Mabs; nz = U[3] / Mabs; }
  W[0] = rho;
  W[1] = g * beta * nx;                                                /* u = gamma v, v = beta M/|M| (Eq. 56) */
  W[2] = g * beta * ny;
  W[3] = g * beta * nz;
  W[4] = (G - 1.0) * (E - beta * Mabs - rho);                          /* Eq. 57 */
  if (!(beta >= 0.0 && beta < 1.0) || !finite5(W) || !(W[4] > 0.0)) return 2;
  return 0;
}

/* (2) Taub-Matthews, ITERATIVE route (:392): Brent's method [36] on the cubic of Eq. 61 in
 * W = gamma^2 - 1, bracketed by gamma in [1, 200] and re-bracketed upwards (gamma -> 10 gamma) while
 * the root is not inside; at most max_iter iterations (the paper's Fig. 2 uses 25 and 50), stopped
 * early when the bracket has shrunk to 4 ulp.  Finishing Eq. 74-75. */
static double tm_cubic(double W, double c1, double c2, double c3) { return ((W + c1) * W + c2) * W + c3; }

static int con2prim_tm_brent(const double U[5], double Wp[5], int max_iter, int *niter_out) {
  double D = U[0], E = U[4];
  double Mabs = sqrt(U[1] * U[1] + U[2] * U[2] + U[3] * U[3]);
  double xi = Mabs / D, eta = E / D;
  double x2 = xi * xi, e2 = eta * eta;
  double dif = (eta - xi) * (eta + xi), den = dif * dif;
  double sum = e2 + x2, br = 4.0 * sum - (x2 + 1.0);
  double c1 = (sum * br - 14.0 * x2 * e2) / (2.0 * den);
  double c2 = (br * br - 57.0 * x2 * e2) / (16.0 * den);
  double c3 = -9.0 * x2 * e2 / (16.0 * den);
  double a = 0.0, b = 200.0 * 200.0 - 1.0;
  double fa = tm_cubic(a, c1, c2, c3), fb = tm_cubic(b, c1, c2, c3);
  for (int k = 0; k < 40 && fb < 0.0; ++k) { b = 100.0 * (b + 1.0) - 1.0; fb = tm_cubic(b, c1, c2, c3); }
  int it = 0;
  double Wv;
  if (fa == 0.0) Wv = a;
  else if (!(fa < 0.0 && fb >= 0.0)) Wv = NAN;
  else {
    /* Brent's method: a = contrapoint, b = best estimate, c = previous b */
    double c = a, fc = fa, d = b - a, e = d;
    for (it = 0; it < max_iter; ++it) {
      if ((fb > 0.0 && fc > 0.0) || (fb < 0.0 && fc < 0.0)) { c = a; fc = fa; d = b - a; e = d; }
      if (fabs(fc) < fabs(fb)) { a = b; b = c; c = a; fa = fb; fb = fc; fc = fa; }
      double tol = 2.0 * 2.220446049250313e-16 * fabs(b), m = 0.5 * (c - b);
      if (fabs(m) <= tol || fb == 0.0) break;
      if (fabs(e) >= tol && fabs(fa) > fabs(fb)) {
        double p, q, s = fb / fa;
        if (a == c) { p = 2.0 * m * s; q = 1.0 - s; }                   /* secant */
        else {                                                          /* inverse quadratic */
          double qq = fa / fc, r = fb / fc;
          p = s * (2.0 * m * qq * (qq - r) - (b - a) * (r - 1.0));
          q = (qq - 1.0) * (r - 1.0) * (s - 1.0);
        }
        if (p > 0.0) q = -q; else p = -p;
        if (2.0 * p < fmin(3.0 * m * q - fabs(tol * q), fabs(e * q))) { e = d; d = p / q; }
        else { d = m; e = m; }
      } else { d = m; e = m; }
      a = b; fa = fb;
      b += (fabs(d) > tol) ? d : (m > 0.0 ? tol : -tol);
      fb = tm_cubic(b, c1, c2, c3);
    }
    Wv = b;
  }
  if (niter_out) *niter_out = it;
  if (Wv < 0.0) Wv = 0.0;
  double g = sqrt(Wv + 1.0), beta = sqrt(Wv / (Wv + 1.0));             /* Eq. 74 */
  double rho = D / g;
  double nx = 0.0, ny = 0.0, nz = 0.0;
  if (Mabs > 0.0) { nx = U[1] / Mabs; ny = U[2] / Mabs; nz = U[3] / Mabs; }
  double ug = sqrt(Wv);
  double X = E - beta * Mabs;
  Wp[0] = rho; Wp[1] = ug * nx; Wp[2] = ug * ny; Wp[3] = ug * nz;
  Wp[4] = (X - rho) * (X + rho) / (3.0 * X);                            /* Eq. 75 */
  if (!finite5(Wp) || !(Wp[4] > 0.0)) return 2;
  return 0;
}

/* variant = 0: the hot-path solvers (orc_con2prim); 1: ideal analytic / Taub-Matthews Brent */
int orc_con2prim_variant(int eos, int variant, double G, const double U[5], double W[5], int max_iter,
                         int *niter_out) {
  if (niter_out) *niter_out = 0;
  if (variant == 0) return orc_con2prim(eos, G, U, W, niter_out);
  if (!orc_admissible(U, 0.0)) {
    for (int v = 0; v < 5; ++v) W[v] = NAN;
    return 1;
  }
  if (eos == ORC_EOS_IDEAL) return con2prim_ideal_analytic(G, U, W);
  return con2prim_tm_brent(U, W, max_iter, niter_out);
}

void orc_con2prim_variant_batch(int eos, int variant, double G, int64_t n, const double *U, double *W,
                                int *status, int max_iter) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double u[5], w[5];
    for (int v = 0; v < 5; ++v) u[v] = U[v * n + i];
    int st = orc_con2prim_variant(eos, variant, G, u, w, max_iter, 0);
    for (int v = 0; v < 5; ++v) W[v * n + i] = w[v];
    if (status) status[i] = st;
  }
}

int orc_con2prim(int eos, double G, const double U[5], double W[5], int *niter_out) {
  if (niter_out) *niter_out = 0;
  if (!orc_admissible(U, 0.0)) {            /* Eq. 25: the solvers are specified on admissible U */
    for (int v = 0; v < 5; ++v) W[v] = NAN;
    return 1;
  }
  if (eos == ORC_EOS_IDEAL) return con2prim_ideal(G, U, W, niter_out, -1);
  return con2prim_tm(U, W);
}

int orc_con2prim_ideal_fixed(double G, const double U[5], double W[5], int niter) {
  return con2prim_ideal(G, U, W, 0, niter);
}

void orc_prim2con_batch(int eos, double G, int64_t n, const double *W, double *U) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double w[5], u[5];
    for (int v = 0; v < 5; ++v) w[v] = W[v * n + i];
    orc_prim2con(eos, G, w, u);
    for (int v = 0; v < 5; ++v) U[v * n + i] = u[v];
  }
}

void orc_con2prim_batch(int eos, double G, int64_t n, const double *U, double *W, int *status) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double w[5], u[5];
    for (int v = 0; v < 5; ++v) u[v] = U[v * n + i];
    int st = orc_con2prim(eos, G, u, w, 0);
    for (int v = 0; v < 5; ++v) W[v * n + i] = w[v];
    if (status) status[i] = st;
  }
}

/* ------------------------------------------------------------------------------------------
 * Mesh helpers
 * ------------------------------------------------------------------------------------------ */
static int ipow(int b, int e) { int r = 1; while (e-- > 0) r *= b; return r; }

int64_t orc_ndof(const orc_config *c) {
  int64_t ne = 1;
  for (int d = 0; d < c->ndim; ++d) ne *= c->nelem[d];
  return ne * ipow(c->order_p + 1, c->ndim);
}

/* ------------------------------------------------------------------------------------------
 * O5  Spatial operator L(U)  (Eq. 15-18; steps in the order of :128-145).
 *   R_i = sum_d (2/h_d)(1/w_{i_d}) [ sum_q w_q D_{q,i_d} F_d(W_{..q..})
 *                                    - (delta_{i_d,p} Fhat_{d,+} - delta_{i_d,0} Fhat_{d,-}) ]
 * GLL collocation: "interpolation to quadrature points" (:132) is the identity in the volume and
 * a gather of the face node on faces, because l_i(+-1) = delta (reading R1).
 * ------------------------------------------------------------------------------------------ */
void orc_rhs(const orc_config *c, const double *U, double *R, int64_t *n_c2p_fail) {
  const int nd = c->ndim, N = c->order_p + 1, nn = ipow(N, nd);
  const int64_t nx = c->nelem[0], ny = nd > 1 ? c->nelem[1] : 1, nz = nd > 2 ? c->nelem[2] : 1;
  const int64_t ne = nx * ny * nz, ndof = ne * nn;
  double x[5], w[5], D[25], h[3];
  orc_gll(N, x, w, D);
  for (int d = 0; d < nd; ++d) h[d] = (c->xmax[d] - c->xmin[d]) / (double)c->nelem[d];
  const int64_t nel[3] = {nx, ny, nz};
  const int str[3] = {1, N, N * N};          /* node stride per direction */

  /* step 1 (Eq. 16): W_i = p(U_i) at every nodal point */
  double *W = (double *)malloc(sizeof(double) * 5 * (size_t)ndof);
  int64_t nfail = 0;
#pragma omp parallel for schedule(static) reduction(+ : nfail)
  for (int64_t i = 0; i < ndof; ++i) {
    double u[5], p[5];
    for (int v = 0; v < 5; ++v) u[v] = U[v * ndof + i];
    if (orc_con2prim(c->eos, c->gamma_ad, u, p, 0) != 0) nfail++;
    for (int v = 0; v < 5; ++v) W[v * ndof + i] = p[v];
  }
  if (n_c2p_fail) *n_c2p_fail += nfail;

#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < ne; ++e) {
    int64_t ie[3] = {e % nx, (e / nx) % ny, e / (nx * ny)};
    /* physical flux at every node of the element, every direction (Eq. 2) */
    double Fe[3][125][5];
    for (int n = 0; n < nn; ++n) {
      double p[5];
      for (int v = 0; v < 5; ++v) p[v] = W[v * ndof + e * nn + n];
      for (int d = 0; d < nd; ++d) orc_flux(c->eos, c->gamma_ad, p, d, Fe[d][n]);
    }
    for (int n = 0; n < nn; ++n) {
      int in[3] = {n % N, (n / N) % N, n / (N * N)};
      double acc[5] = {0, 0, 0, 0, 0};
      for (int d = 0; d < nd; ++d) {
        double term[5] = {0, 0, 0, 0, 0};
        /* volume quadrature, Eq. 17 */
        for (int q = 0; q < N; ++q) {
          int nq = n + (q - in[d]) * str[d];
          for (int v = 0; v < 5; ++v) term[v] += w[q] * D[q * N + in[d]] * Fe[d][nq][v];
        }
        /* surface quadrature, Eq. 18/20 */
        for (int side = 0; side < 2; ++side) {
          if (side == 0 && in[d] != 0) continue;        /* l_i(-1) = delta_{i,0} */
          if (side == 1 && in[d] != N - 1) continue;    /* l_i(+1) = delta_{i,p} */
          int64_t je[3] = {ie[0], ie[1], ie[2]};
          je[d] += side ? 1 : -1;
          int has_nb = 1, bck = ORC_BC_PERIODIC;
          if (je[d] < 0 || je[d] >= nel[d]) {
            const int lo = c->bc[d] & 255, hi = (c->bc[d] >> 8) & 255;
            bck = (side && hi) ? hi : lo;               /* condition at this end of the axis */
            if (bck == ORC_BC_PERIODIC) je[d] = (je[d] + nel[d]) % nel[d];
            else has_nb = 0;                            /* a ghost state stands in for the neighbour */
          }
          int64_t en = je[0] + nx * (je[1] + ny * je[2]);
          int n_nb = n + ((side ? 0 : N - 1) - in[d]) * str[d];   /* neighbour's facing node */
          double Wown[5], Wnb[5], Fh[5];
          for (int v = 0; v < 5; ++v) {
            Wown[v] = W[v * ndof + e * nn + n];
            Wnb[v] = has_nb ? W[v * ndof + en * nn + n_nb] : Wown[v];   /* outflow: own state (R12) */
          }
          if (!has_nb && bck == ORC_BC_REFLECT) Wnb[1 + d] = -Wnb[1 + d];          /* wall */
          if (!has_nb && bck == ORC_BC_DIRICHLET)
            for (int v = 0; v < 5; ++v) Wnb[v] = c->bc_state[d][side][v];           /* fixed state */
          const double *WLp = side ? Wown : Wnb, *WRp = side ? Wnb : Wown;       /* left = lower x_d */
          if (c->riemann == ORC_RIEMANN_HLLC) orc_hllc(c->eos, c->gamma_ad, WLp, WRp, d, Fh, 0, 0, 0);
          else orc_hll(c->eos, c->gamma_ad, WLp, WRp, d, Fh);
          for (int v = 0; v < 5; ++v) term[v] -= side ? Fh[v] : -Fh[v];
        }
        for (int v = 0; v < 5; ++v) acc[v] += (2.0 / h[d]) * (1.0 / w[in[d]]) * term[v];
      }
      for (int v = 0; v < 5; ++v) R[v * ndof + e * nn + n] = acc[v];
    }
  }
  free(W);
}

/* ------------------------------------------------------------------------------------------
 * O7  Physicality-enforcing operator (steps 1-4 of :242-252).
 * ------------------------------------------------------------------------------------------ */
/* Per-node largest smoothing factor s_i = s1*s2 toward an admissible mean Ubar
 * (Eq. 28-37; Eq. 37's root evaluated in the cancellation-free form of reading R14;
 * E is replaced by (1-eps_q)E in the predicate and in c, n, g -- reading R13c). */
double orc_limiter_node_s(const double Ubar[5], const double Ui[5], double eps_q) {
  /* stage 1, Eq. 28-30 */
  double sD = Ui[0] > 0.0 ? 1.0 : Ubar[0] / (Ubar[0] - Ui[0]);
  double sE = Ui[4] > 0.0 ? 1.0 : Ubar[4] / (Ubar[4] - Ui[4]);
  double s1 = fmin(sD, sE);
  double U1[5];
  for (int v = 0; v < 5; ++v) U1[v] = Ubar[v] + s1 * (Ui[v] - Ubar[v]);
  if (orc_admissible(U1, eps_q)) return s1;                         /* step 3(c) */
  /* stage 2, Eq. 31-37 with <A,B> = A_E B_E - A_D B_D - A_M.B_M, E -> (1-eps_q)E */
  double f = 1.0 - eps_q;
  double Eb = f * Ubar[4], E1 = f * U1[4];
  double nb = sqrt(Ubar[0] * Ubar[0] + Ubar[1] * Ubar[1] + Ubar[2] * Ubar[2] + Ubar[3] * Ubar[3]);
  double n1 = sqrt(U1[0] * U1[0] + U1[1] * U1[1] + U1[2] * U1[2] + U1[3] * U1[3]);
  double cc = (Eb - nb) * (Eb + nb);                                /* Eq. 36: <Ubar,Ubar> > 0 */
  double nn = (E1 - n1) * (E1 + n1);                                /* <U1,U1> */
  if (!(nn < 0.0)) return s1;            /* q(U1) >= 0: only D1 <= 0 failed; delta_s handles it */
  double g = Eb * E1 - Ubar[0] * U1[0] - Ubar[1] * U1[1] - Ubar[2] * U1[2] - Ubar[3] * U1[3];
  double r = sqrt(g * g - cc * nn);
  double A = g >= 0.0 ? g + r : -cc * nn / (r - g);
  double s2 = A / (A - nn);                                         /* = Eq. 37's root */
  return s1 * s2;
}

void orc_enforce_physicality(const orc_config *c, double *U, unsigned char *flag, double *s_out,
                             int64_t counters[2]) {
  const int nd = c->ndim, N = c->order_p + 1, nn = ipow(N, nd);
  int64_t ne = 1;
  for (int d = 0; d < nd; ++d) ne *= c->nelem[d];
  const int64_t ndof = ne * nn;
  double x[5], w[5], D[25];
  orc_gll(N, x, w, D);
  int64_t nflag = 0, nbad = 0;
#pragma omp parallel for schedule(static) reduction(+ : nflag, nbad)
  for (int64_t e = 0; e < ne; ++e) {
    /* cell volume average, tensor GLL weights, fixed node order */
    double Ub[5] = {0, 0, 0, 0, 0}, wsum = 0.0;
    int bad = 0;
    for (int n = 0; n < nn; ++n) {
      double wn = w[n % N];
      if (nd > 1) wn *= w[(n / N) % N];
      if (nd > 2) wn *= w[n / (N * N)];
      wsum += wn;
      double u[5];
      for (int v = 0; v < 5; ++v) { u[v] = U[v * ndof + e * nn + n]; Ub[v] += wn * u[v]; }
      if (!orc_admissible(u, 0.5 * c->eps_q)) bad = 1;              /* step 1: screen */
    }
    if (flag) flag[e] = (unsigned char)bad;
    if (!bad) { if (s_out) s_out[e] = 1.0; continue; }
    nflag++;
    for (int v = 0; v < 5; ++v) Ub[v] /= wsum;
    double s = 1.0;
    if (!orc_admissible(Ub, c->eps_q)) {                            /* step 2; R13d */
      nbad++;
      s = 0.0;
    } else {
      for (int n = 0; n < nn; ++n) {                                /* step 3 */
        double u[5];
        for (int v = 0; v < 5; ++v) u[v] = U[v * ndof + e * nn + n];
        double si = orc_limiter_node_s(Ub, u, c->eps_q);
        if (!(si >= 0.0)) si = 0.0;                                 /* NaN guard */
        if (si < s) s = si;                                         /* step 4: s = min s_i */
      }
      s = (1.0 - c->delta_s) * s;                                   /* R13c */
    }
    if (s_out) s_out[e] = s;
    double t = 1.0 - s;
    for (int n = 0; n < nn; ++n)                                    /* Eq. 26, nearer end (R14) */
      for (int v = 0; v < 5; ++v) {
        double ui = U[v * ndof + e * nn + n];
        U[v * ndof + e * nn + n] = (s > 0.5) ? ui + t * (Ub[v] - ui) : Ub[v] + s * (ui - Ub[v]);
      }
  }
  if (counters) { counters[0] += nflag; counters[1] += nbad; }
}

/* ------------------------------------------------------------------------------------------
 * Shock limiter of Moe, Rossmanith & Seal ("the Moe limiter from Moe et al.
 * [23]"; arXiv:1507.03024).  NOT PRINTED IN PAPER.md -- PARITY UNPINNED: this is ref [23]'s algorithm
 * as restated in DESIGN.md reading R18, applied to the five conserved variables w = U:
 *   1. per cell i: average wbar_i (tensor GLL weights) and the extrema w_Mi, w_mi over the cell's
 *      nodes (GLL nodes include the corners and the face points);
 *   2. bounds from the face neighbours N_i (periodic wrap; no neighbour beyond any other boundary):
 *        M_i = max(wbar_i + alpha, max_{j in N_i} w_Mj),  m_i = min(wbar_i - alpha, min_{j in N_i} w_mj);
 *   3. theta_Mi = phi((M_i - wbar_i)/(w_Mi - wbar_i)), theta_mi = phi((m_i - wbar_i)/(w_mi - wbar_i)),
 *      phi(y) = min(y/1.1, 1)  (ratio taken as +inf when the cell's own extremum equals its mean to
 *      rounding, |w_M - wbar| <= 1e-12 max(|w_M|, |w_m|): a uniform cell is never rescaled);
 *   4. theta_i = min(1, theta_M, theta_m over all variables);
 *   5. U <- Ubar_i + theta_i (U - Ubar_i)   (cell averages unchanged; a convex blend of admissible
 *      states, so the physicality operator's result stays admissible).
 * ------------------------------------------------------------------------------------------ */
/* ------------------------------------------------------------------------------------------
 * Minmod limiter (PAPER.md:126 "the minmod limiter [24]", :597; ref [24] = van Leer 1979).  NOT
 * PRINTED IN PAPER.md -- PARITY UNPINNED: restated in DESIGN.md reading R19 as van Leer's minmod
 * slope ratio in the scaling form of the Moe limiter (a convex blend toward the cell average, so
 * the physicality operator's result stays admissible), on the five conserved variables w = U:
 *   1. per cell i: average wbar_i and, per direction d, the cell's linear coefficient
 *        a_d = sum_n w_n xi_d(n) w(n) / sum_n w_n xi_d(n)^2      (tensor GLL weights, xi in [-1,1]:
 *      the linear part of w changes by +-a_d from the cell centre to its faces);
 *   2. neighbour differences D+ = wbar_{i+e_d} - wbar_i, D- = wbar_i - wbar_{i-e_d} (periodic wrap; a
 *      missing neighbour beyond any other boundary drops out of the minmod);
 *   3. limited coefficient  a~_d = minmod(a_d, beta D+/2, beta D-/2)  (beta = 1: van Leer's minmod,
 *      the face value stays within the half difference; beta = 2: the generalised slope limiter of
 *      the RKDG literature [19-22]);  ratio r_d = a~_d / a_d in [0,1]  (1 where |a_d| is zero to
 *      rounding, <= 1e-12 max|w| of the cell);
 *   4. theta_i = min over the variables and directions of r_d, taken as 1 if >= 1 - 1e-12;
 *   5. U <- Ubar_i + theta_i (U - Ubar_i).
 * ------------------------------------------------------------------------------------------ */
static double orc_minmod3(double a, double b, int has_b, double c, int has_c) {
  double s = (a > 0.0) - (a < 0.0), m = fabs(a);
  if (s == 0.0) return 0.0;
  if (has_b) { if (b * s <= 0.0) return 0.0; if (fabs(b) < m) m = fabs(b); }
  if (has_c) { if (c * s <= 0.0) return 0.0; if (fabs(c) < m) m = fabs(c); }
  return s * m;
}

static int64_t orc_minmod_limiter(const orc_config *c, double *U, double *theta_out) {
  const int nd = c->ndim, N = c->order_p + 1, nn = ipow(N, nd);
  const int64_t nx = c->nelem[0], ny = nd > 1 ? c->nelem[1] : 1, nz = nd > 2 ? c->nelem[2] : 1;
  const int64_t ne = nx * ny * nz, ndof = ne * nn;
  const int64_t nel[3] = {nx, ny, nz};
  const double beta = (c->moe_alpha > 0.0) ? c->moe_alpha : 1.0;
  double x[5], w[5], D[25];
  orc_gll(N, x, w, D);
  double *st = (double *)malloc(sizeof(double) * 25 * (size_t)ne);   /* mean[5], a[3][5], max|w|[5] */
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < ne; ++e) {
    double wsum = 0.0, xx[3] = {0, 0, 0}, mean[5] = {0, 0, 0, 0, 0}, a[3][5] = {{0}}, big[5] = {0, 0, 0, 0, 0};
    for (int n = 0; n < nn; ++n) {
      const int idx[3] = {n % N, (n / N) % N, n / (N * N)};
      double wn = w[idx[0]];
      if (nd > 1) wn *= w[idx[1]];
      if (nd > 2) wn *= w[idx[2]];
      wsum += wn;
      for (int d = 0; d < nd; ++d) xx[d] += wn * x[idx[d]] * x[idx[d]];
      for (int v = 0; v < 5; ++v) {
        double u = U[v * ndof + e * nn + n];
        mean[v] += wn * u;
        for (int d = 0; d < nd; ++d) a[d][v] += wn * x[idx[d]] * u;
        if (fabs(u) > big[v]) big[v] = fabs(u);
      }
    }
    for (int v = 0; v < 5; ++v) {
      st[e * 25 + v] = mean[v] / wsum;
      for (int d = 0; d < 3; ++d) st[e * 25 + 5 + 5 * d + v] = (d < nd && N > 1) ? a[d][v] / xx[d] : 0.0;
      st[e * 25 + 20 + v] = big[v];
    }
  }
  int64_t nlim = 0;
#pragma omp parallel for schedule(static) reduction(+ : nlim)
  for (int64_t e = 0; e < ne; ++e) {
    int64_t ie[3] = {e % nx, (e / nx) % ny, e / (nx * ny)};
    double theta = 1.0;
    for (int v = 0; v < 5; ++v) {
      const double wb = st[e * 25 + v], tiny = 1e-12 * st[e * 25 + 20 + v];
      for (int d = 0; d < nd; ++d) {
        const double a = st[e * 25 + 5 + 5 * d + v];
        if (!(fabs(a) > tiny)) continue;
        double dif[2] = {0, 0};
        int has[2] = {0, 0};
        for (int side = 0; side < 2; ++side) {
          int64_t je[3] = {ie[0], ie[1], ie[2]};
          je[d] += side ? 1 : -1;
          if (je[d] < 0 || je[d] >= nel[d]) {
            if ((c->bc[d] & 255) != ORC_BC_PERIODIC) continue;
            je[d] = (je[d] + nel[d]) % nel[d];
          }
          int64_t en = je[0] + nx * (je[1] + ny * je[2]);
          dif[side] = side ? st[en * 25 + v] - wb : wb - st[en * 25 + v];
          has[side] = 1;
        }
        const double al = orc_minmod3(a, 0.5 * beta * dif[1], has[1], 0.5 * beta * dif[0], has[0]);
        const double r = al / a;
        if (r < theta) theta = r;
      }
    }
    if (theta >= 1.0 - 1e-12) theta = 1.0;
    if (theta_out) theta_out[e] = theta;
    if (theta < 1.0) {
      nlim++;
      for (int n = 0; n < nn; ++n)
        for (int v = 0; v < 5; ++v) {
          double ub = st[e * 25 + v];
          U[v * ndof + e * nn + n] = ub + theta * (U[v * ndof + e * nn + n] - ub);
        }
    }
  }
  free(st);
  return nlim;
}

int64_t orc_shock_limiter(const orc_config *c, double *U, double *theta_out) {
  if (c->shock_limiter == 2) return orc_minmod_limiter(c, U, theta_out);
  const int nd = c->ndim, N = c->order_p + 1, nn = ipow(N, nd);
  const int64_t nx = c->nelem[0], ny = nd > 1 ? c->nelem[1] : 1, nz = nd > 2 ? c->nelem[2] : 1;
  const int64_t ne = nx * ny * nz, ndof = ne * nn;
  const int64_t nel[3] = {nx, ny, nz};
  double x[5], w[5], D[25];
  orc_gll(N, x, w, D);
  double *st = (double *)malloc(sizeof(double) * 15 * (size_t)ne);      /* mean, max, min per cell */
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < ne; ++e) {
    double wsum = 0.0, mean[5] = {0, 0, 0, 0, 0}, mx[5], mn[5];
    for (int n = 0; n < nn; ++n) {
      double wn = w[n % N];
      if (nd > 1) wn *= w[(n / N) % N];
      if (nd > 2) wn *= w[n / (N * N)];
      wsum += wn;
      for (int v = 0; v < 5; ++v) {
        double u = U[v * ndof + e * nn + n];
        mean[v] += wn * u;
        if (n == 0 || u > mx[v]) mx[v] = u;
        if (n == 0 || u < mn[v]) mn[v] = u;
      }
    }
    for (int v = 0; v < 5; ++v) { st[e * 15 + v] = mean[v] / wsum; st[e * 15 + 5 + v] = mx[v]; st[e * 15 + 10 + v] = mn[v]; }
  }
  int64_t nlim = 0;
#pragma omp parallel for schedule(static) reduction(+ : nlim)
  for (int64_t e = 0; e < ne; ++e) {
    int64_t ie[3] = {e % nx, (e / nx) % ny, e / (nx * ny)};
    double theta = 1.0;
    for (int v = 0; v < 5; ++v) {
      double wb = st[e * 15 + v], wM = st[e * 15 + 5 + v], wm = st[e * 15 + 10 + v];
      double M = wb + c->moe_alpha, m = wb - c->moe_alpha;
      for (int d = 0; d < nd; ++d)
        for (int side = 0; side < 2; ++side) {
          int64_t je[3] = {ie[0], ie[1], ie[2]};
          je[d] += side ? 1 : -1;
          if (je[d] < 0 || je[d] >= nel[d]) {
            if ((c->bc[d] & 255) != ORC_BC_PERIODIC) continue;
            je[d] = (je[d] + nel[d]) % nel[d];
          }
          int64_t en = je[0] + nx * (je[1] + ny * je[2]);
          if (st[en * 15 + 5 + v] > M) M = st[en * 15 + 5 + v];
          if (st[en * 15 + 10 + v] < m) m = st[en * 15 + 10 + v];
        }
      double tiny = 1e-12 * fmax(fabs(wM), fabs(wm));           /* extremum = mean to rounding: no limit */
      double tM = (wM - wb > tiny) ? fmin((M - wb) / (wM - wb) / 1.1, 1.0) : 1.0;
      double tm = (wb - wm > tiny) ? fmin((wb - m) / (wb - wm) / 1.1, 1.0) : 1.0;
      if (tM < theta) theta = tM;
      if (tm < theta) theta = tm;
    }
    if (theta_out) theta_out[e] = theta;
    if (theta < 1.0) {
      nlim++;
      for (int n = 0; n < nn; ++n)
        for (int v = 0; v < 5; ++v) {
          double ub = st[e * 15 + v];
          U[v * ndof + e * nn + n] = ub + theta * (U[v * ndof + e * nn + n] - ub);
        }
    }
  }
  free(st);
  return nlim;
}

/* ------------------------------------------------------------------------------------------
 * R11  CFL time step ("adaptive time stepping ... to maintain a certain CFL"):
 *   dt = CFL / max_nodes sum_d (2p+1) max(|lambda-_d|,|lambda+_d|)/h_d
 * ------------------------------------------------------------------------------------------ */
double orc_cfl_dt(const orc_config *c, const double *U, double cfl) {
  const int nd = c->ndim;
  const int64_t ndof = orc_ndof(c);
  double h[3];
  for (int d = 0; d < nd; ++d) h[d] = (c->xmax[d] - c->xmin[d]) / (double)c->nelem[d];
  double amax = 0.0;
#pragma omp parallel for schedule(static) reduction(max : amax)
  for (int64_t i = 0; i < ndof; ++i) {
    double u[5], p[5];
    for (int v = 0; v < 5; ++v) u[v] = U[v * ndof + i];
    orc_con2prim(c->eos, c->gamma_ad, u, p, 0);
    double a = 0.0;
    for (int d = 0; d < nd; ++d) {
      double lm, lp;
      orc_wavespeeds(c->eos, c->gamma_ad, p, d, &lm, &lp);
      a += (double)(2 * c->order_p + 1) * fmax(fabs(lm), fabs(lp)) / h[d];
    }
    if (a > amax) amax = a;       /* NaN never wins (comparison false) */
  }
  return cfl / amax;
}

/* ------------------------------------------------------------------------------------------
 * O6  SSP-RK in Shu-Osher form (coefficients: reading R10); the
 * physicality operator after every stage's combine (reading R15).
 *   stage: U_out = a U0 + b (U_s + dt L(U_s)),  (a,b) = (0,1), (3/4,1/4), (1/3,2/3)
 *   SSPRK2 second stage (1/2,1/2).
 * ------------------------------------------------------------------------------------------ */
void orc_step(const orc_config *c, double *U, double dt_in, int nsteps, double *t_inout,
              int64_t counters[3]) {
  const int64_t ndof = orc_ndof(c);
  const size_t nb = sizeof(double) * 5 * (size_t)ndof;
  double *U0 = (double *)malloc(nb), *R = (double *)malloc(nb);
  double A[3], B[3];
  A[0] = 0.0; B[0] = 1.0;
  if (c->rk_stages == 2) { A[1] = 0.5; B[1] = 0.5; }
  else { A[1] = 0.75; B[1] = 0.25; A[2] = 1.0 / 3.0; B[2] = 2.0 / 3.0; }
  for (int step = 0; step < nsteps; ++step) {
    double dt = dt_in > 0.0 ? dt_in : orc_cfl_dt(c, U, -dt_in);
    memcpy(U0, U, nb);
    for (int st = 0; st < c->rk_stages; ++st) {
      int64_t nf = 0, lim[2] = {0, 0};
      orc_rhs(c, U, R, &nf);
#pragma omp parallel for schedule(static)
      for (int64_t i = 0; i < 5 * ndof; ++i) U[i] = A[st] * U0[i] + B[st] * (U[i] + dt * R[i]);
      orc_enforce_physicality(c, U, 0, 0, lim);
      if (c->shock_limiter) orc_shock_limiter(c, U, 0);                /* reading R18 */
      if (counters) { counters[0] += lim[0]; counters[1] += lim[1]; counters[2] += nf; }
    }
    if (t_inout) *t_inout += dt;
  }
  free(U0);
  free(R);
}

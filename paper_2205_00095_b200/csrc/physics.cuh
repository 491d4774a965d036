// physics.cuh -- pointwise relativistic-hydro device functions of the CUDA path (sm_100a, fp64).
//
// Written from PAPER.md (arxiv 2205.00095); shares nothing with oracle/.  Units c = 1.
//   U = [D, Mx, My, Mz, E]  conserved (Eq. 1, Eq. 4);  W = [rho, ux, uy, uz, P], u = gamma v (:47).
// Each function cites the passage it implements.  Arithmetic is arranged for few fp64 divisions
// and square roots (the FP64 pipe is the binding resource of the fused stage kernel);
// FMA contraction is allowed everywhere except in dg_admissible(), which must decide exactly as
// the separately rounded expression of DESIGN.md reading R13e.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#define DG_EOS_IDEAL 0
#define DG_EOS_TM 1
#define DG_INL __device__ __forceinline__

// EOS constants handed to the kernels: G = Gamma, al = Gamma/(Gamma-1) (ideal EOS only).
struct EosPar {
  double G, al;
};

// rho*h as a function of (rho, P):  ideal Eq. 8: rho h = rho + al P;
// Taub-Matthews Eq. 10: rho h = 5/2 P + 3/2 sqrt(P^2 + 4/9 rho^2)   (h(Theta) times rho).
template <int EOS>
DG_INL double dg_rho_h(const EosPar& e, double rho, double P) {
  if (EOS == DG_EOS_IDEAL) return fma(e.al, P, rho);
  return fma(2.5, P, 1.5 * sqrt(fma(P, P, (4.0 / 9.0) * rho * rho)));
}

// sigma_s of Eq. 22, sigma = cs^2 / (gamma^2 (1 - cs^2)), with cs^2 of Eq. 9 / Eq. 11 folded in so
// that only one division remains:
//   ideal: cs^2 = G P/(rho h)          => sigma = G P / (g2 (rho h - G P))
//   TM:    cs^2 = num/den, num = 3 Th^2 + 5 Th r, den = 12 Th^2 + 2 + 12 Th r, r = sqrt(Th^2+4/9),
//          multiply through by rho^2 (R = rho r = sqrt(P^2 + 4/9 rho^2)):
//          sigma = (3 P^2 + 5 P R) / (g2 (9 P^2 + 2 rho^2 + 7 P R))
template <int EOS>
DG_INL double dg_sigma(const EosPar& e, double rho, double P, double g2) {
  if (EOS == DG_EOS_IDEAL) {
    double GP = e.G * P;
    double rh = fma(e.al, P, rho);
    return GP / (g2 * (rh - GP));
  }
  double R = sqrt(fma(P, P, (4.0 / 9.0) * rho * rho));
  double PR = P * R;
  double num = fma(3.0 * P, P, 5.0 * PR);
  double den = fma(9.0 * P, P, fma(2.0 * rho, rho, 7.0 * PR));
  return num / (g2 * den);
}

// Eq. 4: D = gamma rho, M = gamma rho h u, E = gamma^2 rho h - P  with gamma = sqrt(1+|u|^2).
template <int EOS>
DG_INL void dg_prim2con(const EosPar& e, const double W[5], double U[5]) {
  double g2 = fma(W[1], W[1], fma(W[2], W[2], fma(W[3], W[3], 1.0)));
  double g = sqrt(g2);
  double rh = dg_rho_h<EOS>(e, W[0], W[4]);
  double grh = g * rh;
  U[0] = g * W[0];
  U[1] = grh * W[1];
  U[2] = grh * W[2];
  U[3] = grh * W[3];
  U[4] = fma(g2, rh, -W[4]);
}

// Everything a face needs from one side, for direction dir (runtime, 0..2; selects keep W and F in
// registers):
//   U (Eq. 4), F_dir (Eq. 2: F = U v_d + P e_d, F_E = (E+P) v_d) and lambda-+ (Eq. 21-22).
template <int EOS>
DG_INL void dg_side(const EosPar& e, const double W[5], int dir, double U[5], double F[5],
                    double& lm, double& lp) {
  double g2 = fma(W[1], W[1], fma(W[2], W[2], fma(W[3], W[3], 1.0)));
  double rg = rsqrt(g2);
  double g = g2 * rg;
  double rho = W[0], P = W[4];
  double rh = dg_rho_h<EOS>(e, rho, P);
  double grh = g * rh;
  U[0] = g * rho;
  U[1] = grh * W[1];
  U[2] = grh * W[2];
  U[3] = grh * W[3];
  U[4] = fma(g2, rh, -P);
  double ud = (dir == 0) ? W[1] : ((dir == 1) ? W[2] : W[3]);
  double vd = ud * rg;
  F[0] = U[0] * vd;
  F[1] = fma(U[1], vd, (dir == 0) ? P : 0.0);
  F[2] = fma(U[2], vd, (dir == 1) ? P : 0.0);
  F[3] = fma(U[3], vd, (dir == 2) ? P : 0.0);
  F[4] = (U[4] + P) * vd;
  double sig = dg_sigma<EOS>(e, rho, P, g2);
  double root = sqrt(sig * (fma(-vd, vd, 1.0) + sig));
  double r1 = 1.0 / (1.0 + sig);
  lm = (vd - root) * r1;
  lp = (vd + root) * r1;
}

// HLL two-wave flux (PAPER.md:161 cites Schneider et al.; reading R9) with lambda_L,
// lambda_R of Eq. 23-24; U_{L,R} from W_{L,R} by Eq. 4 (reading R8).
template <int EOS>
DG_INL void dg_hll(const EosPar& e, const double WL[5], const double WR[5], int dir, double F[5]) {
  double UL[5], UR[5], FL[5], FR[5], lmL, lpL, lmR, lpR;
  dg_side<EOS>(e, WL, dir, UL, FL, lmL, lpL);
  dg_side<EOS>(e, WR, dir, UR, FR, lmR, lpR);
  double lL = fmin(lmL, lmR);
  double lR = fmax(lpL, lpR);
  if (lL >= 0.0) {
#pragma unroll
    for (int v = 0; v < 5; ++v) F[v] = FL[v];
  } else if (lR <= 0.0) {
#pragma unroll
    for (int v = 0; v < 5; ++v) F[v] = FR[v];
  } else {
    double rd = 1.0 / (lR - lL);
    double ll = lL * lR;
#pragma unroll
    for (int v = 0; v < 5; ++v)
      F[v] = (fma(lR, FL[v], -lL * FR[v]) + ll * (UR[v] - UL[v])) * rd;
  }
}

// sum_d cw[d] max(|lambda-_d|, |lambda+_d|) for the CFL reduction (reading R11, Eq. 21-22).
template <int EOS, int ND>
DG_INL double dg_cfl_speed(const EosPar& e, const double W[5], const double cw[3]) {
  double g2 = fma(W[1], W[1], fma(W[2], W[2], fma(W[3], W[3], 1.0)));
  double rg = rsqrt(g2);
  double sig = dg_sigma<EOS>(e, W[0], W[4], g2);
  double r1 = 1.0 / (1.0 + sig);
  double a = 0.0;
#pragma unroll
  for (int d = 0; d < ND; ++d) {
    double vd = W[1 + d] * rg;
    double root = sqrt(sig * (fma(-vd, vd, 1.0) + sig));
    a = fma(cw[d], (fabs(vd) + root) * r1, a);      // max(|v-r|,|v+r|) = |v| + r  (r >= 0)
  }
  return a;
}

// Admissibility predicate, Eq. 25 with the plus sign (Eq. 27/31/32; reading R13a) and the safety
// factor on E (R13c): D > 0 && (1-eps) E > sqrt(D^2 + Mx^2 + My^2 + Mz^2), every operation rounded
// separately in exactly this order (R13e) so that the decision is bit-identical to the reference
// expression.  NaN anywhere => false.
DG_INL bool dg_admissible(const double U[5], double one_minus_eps) {
  double m2 = __dmul_rn(U[0], U[0]);
  m2 = __dadd_rn(m2, __dmul_rn(U[1], U[1]));
  m2 = __dadd_rn(m2, __dmul_rn(U[2], U[2]));
  m2 = __dadd_rn(m2, __dmul_rn(U[3], U[3]));
  double Es = __dmul_rn(one_minus_eps, U[4]);
  return (U[0] > 0.0) && (Es > __dsqrt_rn(m2));
}

// ---------------------------------------------------------------------------------------------
// con2prim.  Returns status: 0 ok, 1 inadmissible input (W = NaN), 2 P <= 0 or non-finite.
// ---------------------------------------------------------------------------------------------
DG_INL bool dg_finite5(const double W[5]) {
  return isfinite(W[0]) && isfinite(W[1]) && isfinite(W[2]) && isfinite(W[3]) && isfinite(W[4]);
}

// Ideal EOS: Newton on the quartic of Eq. 59 in w, beta = 2w/(1+w^2) (Eq. 58),
// start beta_0 = |M|/E (reading R2), stop |dw| <= 1e-14 w or 16 iterations (R3), small-xi series
// Eq. 60 for xi < 1e-4 (R4); finishing Eq. 55-57 with 1/gamma = (1-w^2)/(1+w^2).
DG_INL int dg_con2prim_ideal(const EosPar& e, const double U[5], double W[5]) {
  const double D = U[0], E = U[4];
  const double M2 = fma(U[1], U[1], fma(U[2], U[2], U[3] * U[3]));
  const double Mabs = sqrt(M2);
  const double xi = Mabs / D, eta = E / D;                       // Eq. 38
  const double al = e.al;
  double w;
  if (xi < 1e-4) {
    if (xi == 0.0) {
      w = 0.0;
    } else {                                                     // Eq. 60
      double a1 = fma(al, eta, -1.0);
      double a12 = a1 * a1;
      double am = al - 1.0;
      double t3 = am * am / (8.0 * a12 * a12) *
                  ((al + 3.0) * fma(al, eta, 1.0) - 4.0 * (al + 1.0));
      w = am / (2.0 * a1) * xi + t3 * xi * xi * xi;
    }
  } else {
    const double c4 = (al - 1.0) * xi;                           // Eq. 59 (c0 = c4)
    const double c3 = -2.0 * fma(al, eta, 1.0);
    const double c2 = 2.0 * (al + 1.0) * xi;
    const double c1 = -2.0 * fma(al, eta, -1.0);
    const double b0 = xi / eta;
    w = b0 / (1.0 + sqrt(fma(-b0, b0, 1.0)));
#pragma unroll 1
    for (int it = 0; it < 16; ++it) {
      double p = fma(fma(fma(fma(c4, w, c3), w, c2), w, c1), w, c4);
      double dp = fma(fma(fma(4.0 * c4, w, 3.0 * c3), w, 2.0 * c2), w, c1);
      double dw = p / dp;
      w -= dw;
      if (fabs(dw) <= 1e-14 * w) break;
    }
  }
  const double w2 = w * w;
  const double r1 = 1.0 / (1.0 + w2);
  const double om = 1.0 - w2;
  const double beta = 2.0 * w * r1;                              // Eq. 58
  const double rho = D * om * r1;                                // Eq. 55, 1/gamma = (1-w^2)/(1+w^2)
  const double ug = 2.0 * w / om;                                // gamma beta
  const double sc = (Mabs > 0.0) ? ug / Mabs : 0.0;              // u = gamma beta M/|M|  (Eq. 56)
  W[0] = rho;
  W[1] = sc * U[1];
  W[2] = sc * U[2];
  W[3] = sc * U[3];
  W[4] = (e.G - 1.0) * (E - beta * Mabs - rho);                  // Eq. 57
  if (!(w >= 0.0 && w < 1.0) || !dg_finite5(W) || !(W[4] > 0.0)) return 2;
  return 0;
}

// Taub-Matthews: cubic in Wv = gamma^2 - 1 with c1..c3 of Eq. 62-64, Q, R, d of
// Eq. 65-67, trigonometric branch Eq. 69-70 (d < 0) or Cardano Eq. 71-73 (d >= 0), then Eq. 74-75.
// Safeguards of reading R7: eta^2-xi^2 = (eta-xi)(eta+xi), acos argument clamped, Wv >= 0; R7b: one
// Newton correction of the root on the cubic itself (full relative accuracy as gamma -> 1).
DG_INL int dg_con2prim_tm(const double U[5], double W[5]) {
  const double D = U[0], E = U[4];
  const double M2 = fma(U[1], U[1], fma(U[2], U[2], U[3] * U[3]));
  const double Mabs = sqrt(M2);
  const double xi = Mabs / D, eta = E / D;                       // Eq. 38
  const double x2 = xi * xi, e2 = eta * eta;
  const double dif = (eta - xi) * (eta + xi);
  const double rden = 1.0 / (dif * dif);
  const double sum = e2 + x2;
  const double br = 4.0 * sum - (x2 + 1.0);
  const double xe = x2 * e2;
  const double c1 = (sum * br - 14.0 * xe) * (0.5 * rden);       // Eq. 62
  const double c2 = (br * br - 57.0 * xe) * (0.0625 * rden);     // Eq. 63
  const double c3 = -9.0 * xe * (0.0625 * rden);                 // Eq. 64
  const double Q = (3.0 * c2 - c1 * c1) * (1.0 / 9.0);           // Eq. 66
  const double R = (9.0 * c1 * c2 - 27.0 * c3 - 2.0 * c1 * c1 * c1) * (1.0 / 54.0);   // Eq. 67
  const double Q3 = Q * Q * Q;
  const double d = fma(R, R, Q3);                                // Eq. 65
  double Wv;
  if (d < 0.0) {
    double arg = R * rsqrt(-Q3);
    arg = fmin(1.0, fmax(-1.0, arg));
    Wv = 2.0 * sqrt(-Q) * cos(acos(arg) * (1.0 / 3.0)) - c1 * (1.0 / 3.0);   // Eq. 69-70
  } else {
    double sd = sqrt(d);
    Wv = cbrt(R + sd) + cbrt(R - sd) - c1 * (1.0 / 3.0);         // Eq. 71-73
  }
  Wv = fmax(Wv, 0.0);
  {                                                              // R7b: one Newton step on Eq. 61
    const double f = fma(fma(Wv + c1, Wv, c2), Wv, c3);
    const double df = fma(fma(3.0, Wv, 2.0 * c1), Wv, c2);
    const double Wn = Wv - f / df;
    if (isfinite(Wn)) Wv = Wn;
    Wv = fmax(Wv, 0.0);
  }
  const double g2 = Wv + 1.0;
  const double rg = rsqrt(g2);                                   // 1/gamma, Eq. 74
  const double ug = sqrt(Wv);                                    // gamma beta
  const double beta = ug * rg;
  const double rho = D * rg;
  const double sc = (Mabs > 0.0) ? ug / Mabs : 0.0;
  const double X = fma(-beta, Mabs, E);                          // E - M.v
  W[0] = rho;
  W[1] = sc * U[1];
  W[2] = sc * U[2];
  W[3] = sc * U[3];
  W[4] = (X - rho) * (X + rho) / (3.0 * X);                      // Eq. 75
  if (!dg_finite5(W) || !(W[4] > 0.0)) return 2;
  return 0;
}

template <int EOS>
DG_INL int dg_con2prim(const EosPar& e, const double U[5], double W[5]) {
  if (!dg_admissible(U, 1.0)) {                                  // Eq. 25: solvers need admissible U
    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
#pragma unroll
    for (int v = 0; v < 5; ++v) W[v] = qnan;
    return 1;
  }
  if (EOS == DG_EOS_IDEAL) return dg_con2prim_ideal(e, U, W);
  return dg_con2prim_tm(U, W);
}

// ---------------------------------------------------------------------------------------------
// Physicality operator, per node (Eq. 28-37): largest s = s1 s2 in [0,1] such
// that Ubar + s (U_i - Ubar) is admissible.  Stage 2's root (Eq. 37) is evaluated in the
// cancellation-free form of reading R14 with the Minkowski form <A,B> = A_E B_E - A_D B_D - A_M.B_M
// and E -> (1-eps_q) E (R13c).
// ---------------------------------------------------------------------------------------------
DG_INL double dg_limiter_node_s(const double Ub[5], const double Ui[5], double f /* 1-eps_q */) {
  double sD = (Ui[0] > 0.0) ? 1.0 : Ub[0] / (Ub[0] - Ui[0]);     // Eq. 28
  double sE = (Ui[4] > 0.0) ? 1.0 : Ub[4] / (Ub[4] - Ui[4]);     // Eq. 29
  double s1 = fmin(sD, sE);                                      // Eq. 30
  double U1[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) U1[v] = __dadd_rn(Ub[v], __dmul_rn(s1, __dadd_rn(Ui[v], -Ub[v])));
  if (dg_admissible(U1, f)) return s1;
  double Eb = f * Ub[4], E1 = f * U1[4];
  double nb = sqrt(fma(Ub[0], Ub[0], fma(Ub[1], Ub[1], fma(Ub[2], Ub[2], Ub[3] * Ub[3]))));
  double n1 = sqrt(fma(U1[0], U1[0], fma(U1[1], U1[1], fma(U1[2], U1[2], U1[3] * U1[3]))));
  double cc = (Eb - nb) * (Eb + nb);                             // Eq. 36: <Ubar,Ubar>
  double nn = (E1 - n1) * (E1 + n1);                             // <U1,U1>
  if (!(nn < 0.0)) return s1;
  double g = Eb * E1 - Ub[0] * U1[0] - Ub[1] * U1[1] - Ub[2] * U1[2] - Ub[3] * U1[3];
  double r = sqrt(fma(g, g, -cc * nn));
  double A = (g >= 0.0) ? g + r : -cc * nn / (r - g);
  return s1 * (A / (A - nn));                                    // Eq. 37's root
}

// ordered-integer image of a non-negative double (monotone), for atomicMax / atomicMin
DG_INL unsigned long long dg_ord(double x) { return (unsigned long long)__double_as_longlong(x); }
DG_INL double dg_unord(unsigned long long k) { return __longlong_as_double((long long)k); }

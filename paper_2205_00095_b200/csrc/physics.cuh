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

// Branch-free fp64 reciprocal, reciprocal square root and square root: the MUFU seed
// (rcp/rsqrt.approx.ftz.f64, ~2^-22 relative) refined by two Newton steps (error -> 2^-44 -> below one
// ulp), without the denormal/overflow slow paths of the IEEE sequences.  Results are within ~1 ulp
// of the correctly rounded ones -- far inside every tolerance of this path; the one place where the
// decision must be bit-exact (dg_admissible) does not use them.  Arguments are positive, normal
// numbers on every admissible state.
DG_INL double dg_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  r = fma(r, fma(-x, r, 1.0), r);
  r = fma(r, fma(-x, r, 1.0), r);
  return r;
}
DG_INL double dg_rsqrt(double x) {
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double h = 0.5 * x;
  r = fma(r, fma(-h * r, r, 0.5), r);
  r = fma(r, fma(-h * r, r, 0.5), r);
  return r;
}
DG_INL double dg_sqrt(double x) {                 // x >= 0; sqrt(0) = 0
  const double r = dg_rsqrt(fmax(x, 1e-300));
  const double s = x * r;
  return fma(fma(-s, s, x), 0.5 * r, s);
}

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

// sigma_s = num/den of Eq. 22 as an unevaluated fraction (same algebra as dg_sigma).
template <int EOS>
DG_INL void dg_sigma_frac(const EosPar& e, double rho, double P, double g2, double& num, double& den) {
  if (EOS == DG_EOS_IDEAL) {
    num = e.G * P;
    den = g2 * (fma(e.al, P, rho) - num);
  } else {
    const double R = sqrt(fma(P, P, (4.0 / 9.0) * rho * rho));
    const double PR = P * R;
    num = fma(3.0 * P, P, 5.0 * PR);
    den = g2 * fma(9.0 * P, P, fma(2.0 * rho, rho, 7.0 * PR));
  }
}

// lambda-+ of Eq. 21 with sigma = num/den substituted, as fractions over the common positive
// denominator dn = den + num:   lambda-+ = (v den -+ sqrt(num ((1 - v^2) den + num))) / (den + num).
template <int EOS>
DG_INL void dg_speeds_frac(const EosPar& e, double rho, double P, double g2, double vd, double& nm,
                           double& np, double& dn) {
  double num, den;
  dg_sigma_frac<EOS>(e, rho, P, g2, num, den);
  const double root = dg_sqrt(num * fma(fma(-vd, vd, 1.0), den, num));
  const double c = vd * den;
  nm = c - root;
  np = c + root;
  dn = den + num;
}

// One side's contribution to the interface flux:  acc += cF F_dir(W) + cU U(W)   (Eq. 2, Eq. 4).
template <int EOS, int dir>
DG_INL void dg_side_accum(const EosPar& e, const double W[5], double g2, double rg, double vd,
                          double cF, double cU, double acc[5]) {
  const double rho = W[0], P = W[4];
  const double rh = dg_rho_h<EOS>(e, rho, P);
  const double g = g2 * rg;
  const double grh = g * rh;
  const double k = fma(cF, vd, cU);                 // cF U v_d + cU U = U (cF v_d + cU)
  const double cP = cF * P;
  acc[0] = fma(k, g * rho, acc[0]);
  acc[1] = fma(k, grh * W[1], acc[1] + ((dir == 0) ? cP : 0.0));
  acc[2] = fma(k, grh * W[2], acc[2] + ((dir == 1) ? cP : 0.0));
  acc[3] = fma(k, grh * W[3], acc[3] + ((dir == 2) ? cP : 0.0));
  const double E = fma(g2, rh, -P);
  acc[4] = fma(k, E, fma(cP, vd, acc[4]));          // cF (E+P) v_d + cU E
}

// HLL two-wave flux (PAPER.md:161 cites Schneider et al.; reading R9) with lambda_L,
// lambda_R of Eq. 23-24; U_{L,R} from W_{L,R} by Eq. 4 (reading R8).  Branch-free: the three cases
// of R9 are the coefficient triples (1,0,0), (0,1,0), (lR,-lL,lL lR)/(lR-lL) of
//   F = cL F_L + cR F_R + cU (U_R - U_L).
template <int EOS, int dir>
DG_INL void dg_hll(const EosPar& e, const double WL[5], const double WR[5], double F[5]) {
  const double g2L = fma(WL[1], WL[1], fma(WL[2], WL[2], fma(WL[3], WL[3], 1.0)));
  const double g2R = fma(WR[1], WR[1], fma(WR[2], WR[2], fma(WR[3], WR[3], 1.0)));
  const double rgL = dg_rsqrt(g2L), rgR = dg_rsqrt(g2R);
  const double vL = WL[1 + dir] * rgL, vR = WR[1 + dir] * rgR;
  double nmL, npL, dL, nmR, npR, dR;
  dg_speeds_frac<EOS>(e, WL[0], WL[4], g2L, vL, nmL, npL, dL);
  dg_speeds_frac<EOS>(e, WR[0], WR[4], g2R, vR, nmR, npR, dR);
  // lambda_L = min(nmL/dL, nmR/dR) =: nl/dl, lambda_R = max(npL/dL, npR/dR) =: nr/dr  (Eq. 23-24),
  // compared by cross-multiplication (dL, dR > 0); the HLL weights then need one division:
  //   (cL, cR, cU) = (nr dl, -nl dr, nl nr) / (nr dl - nl dr).
  const bool ml = nmL * dR <= nmR * dL, mr = npL * dR >= npR * dL;
  const double nl = ml ? nmL : nmR, dl = ml ? dL : dR;
  const double nr = mr ? npL : npR, dr = mr ? dL : dR;
  double cL, cR, cU;
  if (nl >= 0.0) { cL = 1.0; cR = 0.0; cU = 0.0; }
  else if (nr <= 0.0) { cL = 0.0; cR = 1.0; cU = 0.0; }
  else {
    const double a = nr * dl, b = nl * dr;
    const double q = dg_rcp(a - b);
    cL = a * q; cR = -b * q; cU = nl * nr * q;
  }
#pragma unroll
  for (int v = 0; v < 5; ++v) F[v] = 0.0;
  dg_side_accum<EOS, dir>(e, WL, g2L, rgL, vL, cL, -cU, F);
  dg_side_accum<EOS, dir>(e, WR, g2R, rgR, vR, cR, cU, F);
}

// sum_d cw[d] max(|lambda-_d|, |lambda+_d|) for the CFL reduction (reading R11, Eq. 21-22).
template <int EOS, int ND>
DG_INL double dg_cfl_speed(const EosPar& e, const double W[5], const double cw[3]) {
  const double g2 = fma(W[1], W[1], fma(W[2], W[2], fma(W[3], W[3], 1.0)));
  const double rg = dg_rsqrt(g2);
  double num, den;
  dg_sigma_frac<EOS>(e, W[0], W[4], g2, num, den);
  const double r1 = dg_rcp(den + num);
  double a = 0.0;
#pragma unroll
  for (int d = 0; d < ND; ++d) {
    const double vd = W[1 + d] * rg;
    const double root = dg_sqrt(num * fma(fma(-vd, vd, 1.0), den, num));
    a = fma(cw[d], fma(fabs(vd), den, root), a);    // max(|l-|,|l+|) (den+num) = |v| den + root
  }
  return a * r1;
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
  const double Es = __dmul_rn(one_minus_eps, U[4]);
  if (!(U[0] > 0.0) || !(Es > 0.0)) return false;
  // The decision Es > sqrt(m2) is taken without the square root wherever Es^2 and m2 differ by
  // more than 1e-12 relative (>> the 2-ulp rounding of Es*Es); only marginal states pay for the
  // correctly rounded sqrt, so the result is identical to the reference expression in every case.
  const double t = __dmul_rn(Es, Es);
  if (!(t > 1e-280 && t < 1e300)) return Es > __dsqrt_rn(m2);   // outside the safely normal range
  if (t > __dmul_rn(m2, 1.0 + 1e-12)) return true;
  if (!(t >= __dmul_rn(m2, 1.0 - 1e-12))) return false;
  return Es > __dsqrt_rn(m2);
}

// ---------------------------------------------------------------------------------------------
// con2prim.  Returns status: 0 ok, 1 inadmissible input (W = NaN), 2 P <= 0 or non-finite.
// ---------------------------------------------------------------------------------------------
DG_INL bool dg_finite5(const double W[5]) {
  return isfinite(W[0]) && isfinite(W[1]) && isfinite(W[2]) && isfinite(W[3]) && isfinite(W[4]);
}

// single-precision reciprocal / square root of a double (MUFU): only where the result feeds a
// self-correcting iteration (Newton's step size, its starting point), never a final value.
DG_INL double dg_rcp_lo(double x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(__double2float_rn(x)));
  return (double)r;
}
DG_INL double dg_sqrt_lo(double x) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(__double2float_rn(x)));
  return (double)r;
}

// Ideal EOS: Newton on the quartic of Eq. 59 in w, beta = 2w/(1+w^2) (Eq. 58),
// start beta_0 = |M|/E (reading R2), stop |dw| <= 1e-14 w or 16 iterations (R3), small-xi series
// Eq. 60 for xi < 1e-4 (R4); finishing Eq. 55-57 with 1/gamma = (1-w^2)/(1+w^2).
// fp64 divisions are the expensive operation here, so: xi, eta share 1/D; the Newton step p/p' and
// the starting point use single-precision reciprocals (the iteration corrects them: a step with
// relative error 6e-8 still contracts the error by that factor, and the stopping test is on the
// fp64 step); the three divisions of the finishing formulas share one reciprocal.
DG_INL int dg_con2prim_ideal(const EosPar& e, const double U[5], double W[5]) {
  const double D = U[0], E = U[4];
  const double M2 = fma(U[1], U[1], fma(U[2], U[2], U[3] * U[3]));
  const double Mabs = dg_sqrt(M2);
  const double rD = dg_rcp(D);
  const double xi = Mabs * rD, eta = E * rD;                     // Eq. 38
  const double al = e.al;
  if (xi == 0.0) {                                               // v = 0 (R4)
    W[0] = D; W[1] = 0.0; W[2] = 0.0; W[3] = 0.0;
    W[4] = (e.G - 1.0) * (E - D);
    return (isfinite(W[4]) && W[4] > 0.0) ? 0 : 2;
  }
  double w;
  if (xi < 1e-4) {                                               // Eq. 60
    double a1 = fma(al, eta, -1.0);
    double a12 = a1 * a1;
    double am = al - 1.0;
    double t3 = am * am / (8.0 * a12 * a12) * ((al + 3.0) * fma(al, eta, 1.0) - 4.0 * (al + 1.0));
    w = am / (2.0 * a1) * xi + t3 * xi * xi * xi;
  } else {
    const double c4 = (al - 1.0) * xi;                           // Eq. 59 (c0 = c4)
    const double c3 = -2.0 * fma(al, eta, 1.0);
    const double c2 = 2.0 * (al + 1.0) * xi;
    const double c1 = -2.0 * fma(al, eta, -1.0);
    const double d3 = 4.0 * c4, d2 = 3.0 * c3, d1 = 2.0 * c2;   // p'(w) coefficients
    const bool lo_ok = (eta < 1e30);                             // single-precision range of p'
    if (lo_ok) {
      const double b0 = fmin(xi * dg_rcp_lo(eta), 1.0);
      w = fmin(b0 * dg_rcp_lo(1.0 + dg_sqrt_lo(fmax(fma(-b0, b0, 1.0), 0.0))), 0.999999);
    } else {
      const double b0 = xi / eta;
      w = b0 / (1.0 + sqrt(fma(-b0, b0, 1.0)));
    }
#pragma unroll 1
    for (int it = 0; it < 16; ++it) {
      const double p = fma(fma(fma(fma(c4, w, c3), w, c2), w, c1), w, c4);
      const double dp = fma(fma(fma(d3, w, d2), w, d1), w, c1);
      const double dw = lo_ok ? p * dg_rcp_lo(dp) : p / dp;
      w -= dw;
      if (fabs(dw) <= 1e-14 * w) break;
    }
  }
  const double w2 = w * w;
  const double op = 1.0 + w2, om = 1.0 - w2;
  const double r = dg_rcp(op * om * Mabs);                       // one reciprocal for Eq. 55-58
  const double r1 = r * om * Mabs;                               // 1/(1+w^2)
  const double beta = 2.0 * w * r1;                              // Eq. 58
  const double rho = D * om * r1;                                // Eq. 55, 1/gamma = (1-w^2)/(1+w^2)
  const double sc = 2.0 * w * op * r;                            // gamma beta / |M|  (Eq. 56)
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
  const double Mabs = dg_sqrt(M2);
  const double rD = dg_rcp(D);
  const double xi = Mabs * rD, eta = E * rD;                       // Eq. 38
  const double x2 = xi * xi, e2 = eta * eta;
  const double dif = (eta - xi) * (eta + xi);
  const double rden = dg_rcp(dif * dif);
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
  // The transcendental part of the closed form (acos/cos, Eq. 69-70; cube roots, Eq. 71-73) is
  // evaluated in single precision -- it only has to land in the basin of the wanted root -- and the
  // root is then refined on the cubic of Eq. 61 itself by three Newton steps (reading R7b: the first
  // squares the ~1e-7 seed error, the second reaches the fp64 floor for all gamma, the third covers
  // gamma -> 1 where W = gamma^2-1 is tiny against the seed's absolute error).
  double Wv;
  if (d < 0.0) {
    double arg = R * dg_rsqrt(-Q3);
    arg = fmin(1.0, fmax(-1.0, arg));
    const float th = acosf((float)arg) * (1.0f / 3.0f);
    Wv = 2.0 * dg_sqrt(-Q) * (double)__cosf(th) - c1 * (1.0 / 3.0);        // Eq. 69-70
  } else {
    const double sd = dg_sqrt(d);
    const double p = R + sd, q = R - sd;
    const double cp = (fabs(p) < 1e37) ? (double)cbrtf((float)p) : cbrt(p);
    const double cq = (fabs(q) < 1e37) ? (double)cbrtf((float)q) : cbrt(q);
    Wv = cp + cq - c1 * (1.0 / 3.0);                                       // Eq. 71-73
  }
  Wv = fmax(Wv, 0.0);
#pragma unroll
  for (int it = 0; it < 3; ++it) {                                         // R7b: Newton on Eq. 61
    const double f = fma(fma(Wv + c1, Wv, c2), Wv, c3);
    const double df = fma(fma(3.0, Wv, 2.0 * c1), Wv, c2);
    const double Wn = Wv - f * dg_rcp(df);
    if (isfinite(Wn)) Wv = Wn;
    Wv = fmax(Wv, 0.0);
  }
  const double g2 = Wv + 1.0;
  const double rg = dg_rsqrt(g2);                                  // 1/gamma, Eq. 74
  const double ug = dg_sqrt(Wv);                                   // gamma beta
  const double beta = ug * rg;
  const double rho = D * rg;
  const double sc = (Mabs > 0.0) ? ug * dg_rcp(Mabs) : 0.0;
  const double X = fma(-beta, Mabs, E);                          // E - M.v
  W[0] = rho;
  W[1] = sc * U[1];
  W[2] = sc * U[2];
  W[3] = sc * U[3];
  W[4] = (X - rho) * (X + rho) * dg_rcp(3.0 * X);                      // Eq. 75
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

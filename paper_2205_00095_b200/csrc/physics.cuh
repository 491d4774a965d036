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

// Opt-in debug build (-DDG_DEBUG_ASSERTS): bounds / ownership checks on every shared-memory slot
// index and halo offset of the fused kernel -- the stand-in for compute-sanitizer, which is closed
// on this GPU pool.  A failed check traps the kernel.
#ifdef DG_DEBUG_ASSERTS
#define DG_ASSERT(c) do { if (!(c)) { printf("DG_ASSERT %s:%d: %s\n", __FILE__, __LINE__, #c); __trap(); } } while (0)
#else
#define DG_ASSERT(c) do { } while (0)
#endif

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
// sqrt(x + 1e-300): one add instead of the compare-and-select guard; identical to dg_sqrt(x) for every
// normal x and 1e-150 instead of 0 at x = 0 -- used where that is harmless (|M|, wave-speed radicands).
// One Newton step on the reciprocal root (seed 2^-22 -> 2^-44) is enough here: the closing correction
// s + (y - s^2) r/2 is itself a Newton step for the root and squares the error once more.
DG_INL double dg_sqrt_p(double x) {
  const double y = x + 1e-300;
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(y));
  r = fma(r, fma(-0.5 * y * r, r, 0.5), r);
  const double s = y * r;
  return fma(fma(-s, s, y), 0.5 * r, s);
}

// rho*h as a function of (rho, P):  ideal Eq. 8: rho h = rho + al P;
// Taub-Matthews Eq. 10: rho h = 5/2 P + 3/2 sqrt(P^2 + 4/9 rho^2)   (h(Theta) times rho).
template <int EOS>
DG_INL double dg_rho_h(const EosPar& e, double rho, double P) {
  if (EOS == DG_EOS_IDEAL) return fma(e.al, P, rho);
  return fma(2.5, P, 1.5 * sqrt(fma(P, P, (4.0 / 9.0) * rho * rho)));
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

// What the flux and the wave speeds need at a node, from its conserved state U and its pressure
// P = P(U) (recovered once per node by the stage that produced U and kept in HBM, 8 B per node):
//   r = 1/(E + P);  3-velocity  v = M r        (Eq. 4: M = gamma^2 rho h v, E + P = gamma^2 rho h),
//   q = 1 - |v|^2 = 1/gamma^2,   rho h = (E + P) q,
//   sigma_s = cs^2 / (gamma^2 (1 - cs^2)) of Eq. 22 as an unevaluated fraction num/den:
//     ideal (Eq. 9, cs^2 = G P/(rho h)):   num = G P q,  den = rho h - G P;
//     Taub-Matthews (Eq. 11 times rho^2, R := rho sqrt(Theta^2 + 4/9) = (2 rho h - 5 P)/3 by Eq. 10,
//     rho^2 = 9/4 (R^2 - P^2)):            num = (3 P^2 + 5 P R) q,  den = 9/2 (P^2 + R^2) + 7 P R.
// No square root and one reciprocal; rho itself is never needed.  The flux of Eq. 2 in direction d is
//   F_d = [D v_d, M v_d + P e_d, (E + P) v_d] = [D v_d, M v_d + P e_d, M_d].
template <int EOS>
DG_INL void dg_sigma_r(const EosPar& e, const double U[5], double P, double r, double& num, double& den) {
  const double m2 = fma(U[1], U[1], fma(U[2], U[2], U[3] * U[3]));
  const double q = fma(-r * r, m2, 1.0);
  const double rh = (U[4] + P) * q;
  if (EOS == DG_EOS_IDEAL) {
    const double GP = e.G * P;
    num = GP * q;
    den = rh - GP;
  } else {
    const double R = fma(2.0, rh, -5.0 * P) * (1.0 / 3.0);
    const double PR = P * R;
    num = fma(3.0 * P, P, 5.0 * PR) * q;
    den = fma(4.5, fma(P, P, R * R), 7.0 * PR);
  }
}
template <int EOS>
DG_INL void dg_derive(const EosPar& e, const double U[5], double P, double v[3], double& num, double& den) {
  const double r = dg_rcp(U[4] + P);
  v[0] = U[1] * r; v[1] = U[2] * r; v[2] = U[3] * r;
  dg_sigma_r<EOS>(e, U, P, r, num, den);
}

// lambda-+ of Eq. 21 with sigma = num/den substituted, as fractions over the common positive
// denominator dn = den + num:   lambda-+ = (v den -+ sqrt(num ((1 - v^2) den + num))) / (den + num).
DG_INL void dg_speeds_frac(double vn, double num, double den, double& nm, double& np, double& dn) {
  const double root = dg_sqrt_p(num * fma(fma(-vn, vn, 1.0), den, num));
  const double c = vn * den;
  nm = c - root;
  np = c + root;
  dn = den + num;
}

// sum_d cw[d] max(|lambda-_d|, |lambda+_d|) for the CFL reduction (reading R11, Eq. 21-22), from the
// node's conserved state and pressure.
template <int EOS, int ND>
DG_INL double dg_cfl_speed(const EosPar& e, const double U[5], double P, const double cw[3]) {
  double v[3], num, den;
  dg_derive<EOS>(e, U, P, v, num, den);
  const double r1 = dg_rcp(den + num);
  double a = 0.0;
#pragma unroll
  for (int d = 0; d < ND; ++d) {
    const double root = dg_sqrt_p(num * fma(fma(-v[d], v[d], 1.0), den, num));
    a = fma(cw[d], fma(fabs(v[d]), den, root), a);   // max(|l-|,|l+|) (den+num) = |v| den + root
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
  // The decision Es > sqrt(m2) is taken without the square root wherever Es^2 and m2 differ by
  // more than 1e-12 relative (>> the 2-ulp rounding of Es*Es) and Es^2 is safely normal: one test for
  // the common, clearly admissible case; only marginal or inadmissible states take the exact path, so
  // the result is identical to the reference expression in every case.
  const double t = __dmul_rn(Es, Es);
  if ((U[0] > 0.0) & (Es > 0.0) & (t > __dmul_rn(m2, 1.0 + 1e-12)) & (t > 1e-280) & (t < 1e300)) return true;
  if (!(U[0] > 0.0) || !(Es > 0.0)) return false;
  if (!(t > 1e-280 && t < 1e300)) return Es > __dsqrt_rn(m2);   // outside the safely normal range
  if (!(t >= __dmul_rn(m2, 1.0 - 1e-12))) return false;
  return Es > __dsqrt_rn(m2);
}

// ---------------------------------------------------------------------------------------------
// con2prim.  Status per state: 0 ok, 1 inadmissible input (outputs NaN), 2 P <= 0 or non-finite.
// The solvers work on NS states of one thread in lockstep (NS independent fp64 instruction
// streams: the iteration is latency-bound on one state); a state that has converged is frozen, so
// every state takes exactly the iterates it would take alone.
// ---------------------------------------------------------------------------------------------
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

// Ideal EOS: the root w in (0,1) of the quartic of Eq. 59, beta = 2w/(1+w^2)
// (Eq. 58), by Newton's iteration from beta_0 = |M|/E (reading R2), stopped at |dw| <= 1e-14 w or 16
// iterations (R3); small-xi series Eq. 60 for xi < 1e-4 (R4).  fp64 divisions are the expensive
// operation, so xi and eta share 1/D, and the Newton step p/p' and the starting point are formed in
// single precision (the iteration corrects them: a step with relative error 6e-8 still contracts the
// error by that factor, and the stopping test is on the fp64 step).  States outside the single-
// precision range (eta >= 1e30) or on the series branch take the out-of-line general routine.
// In: D, E, |M| of admissible states.  Out: w.
static __device__ __noinline__ double dg_ideal_w_general(double al, double xi, double eta) {
  if (xi < 1e-4) {                                                 // Eq. 60 (xi = 0 gives w = 0: v = 0)
    const double a1 = fma(al, eta, -1.0);
    const double a12 = a1 * a1;
    const double am = al - 1.0;
    const double t3 = am * am / (8.0 * a12 * a12) * ((al + 3.0) * fma(al, eta, 1.0) - 4.0 * (al + 1.0));
    return am / (2.0 * a1) * xi + t3 * xi * xi * xi;
  }
  const double c4 = (al - 1.0) * xi, c3 = -2.0 * fma(al, eta, 1.0), c2 = 2.0 * (al + 1.0) * xi,
               c1 = -2.0 * fma(al, eta, -1.0);
  const double b0 = xi / eta;
  double w = b0 / (1.0 + sqrt(fma(-b0, b0, 1.0)));
  for (int it = 0; it < 16; ++it) {
    const double p = fma(fma(fma(fma(c4, w, c3), w, c2), w, c1), w, c4);
    const double dp = fma(fma(fma(4.0 * c4, w, 3.0 * c3), w, 2.0 * c2), w, c1);
    const double dw = p / dp;
    w -= dw;
    if (fabs(dw) <= 1e-14 * w) break;
  }
  return w;
}

// Pg (or NULL): a guess of the pressure (the stage kernel passes the pressure of the node's previous
// state): beta_0 = |M| / (E + Pg) instead of |M| / E.  Any start in (0,1) converges.
// Stopping: Newton converges quadratically and the step is a tight estimate of the error BEFORE the
// step, so once |dw| <= 1e-9 w the new iterate is at the fp64 floor (error ~ K dw^2 + 6e-8 |dw| from the
// single-precision reciprocal); this meets reading R3's criterion (|dw| <= 1e-14 w) one iteration earlier.
template <int NS>
DG_INL void dg_ideal_solve_w(const EosPar& e, const double* D, const double* E, const double* Mabs,
                             const double* Pg, double* w) {
  const double al = e.al;
  double c4[NS], c3[NS], c2[NS], c1[NS], xi[NS], eta[NS];
  bool run[NS], general[NS];
  bool any = false;
#pragma unroll
  for (int s = 0; s < NS; ++s) {
    const double rD = dg_rcp(D[s]);
    xi[s] = Mabs[s] * rD; eta[s] = E[s] * rD;                      // Eq. 38
    c4[s] = (al - 1.0) * xi[s];                                    // Eq. 59 (c0 = c4)
    c3[s] = -2.0 * fma(al, eta[s], 1.0);
    c2[s] = 2.0 * (al + 1.0) * xi[s];
    c1[s] = -2.0 * fma(al, eta[s], -1.0);
    // (E or |M| outside the single-precision range only degrades the starting point: 0 or 0.999999)
    general[s] = !(eta[s] < 1e30) || !(xi[s] >= 1e-4);
    run[s] = !general[s];
    // starting point in single precision: b0 = xi/eta, w0 = b0 / (1 + sqrt(1 - b0^2))
    const float xf = __double2float_rn(Mabs[s]);
    const float ef = __double2float_rn(Pg ? E[s] + fmax(Pg[s], 0.0) : E[s]);
    const float b0 = fminf(__fdividef(xf, ef), 1.0f);
    float sq;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(sq) : "f"(fmaxf(fmaf(-b0, b0, 1.0f), 0.0f)));
    const float w0 = fminf(__fdividef(b0, 1.0f + sq), 0.999999f);
    w[s] = (double)w0;
    any = any || run[s];
  }
#pragma unroll 1
  for (int it = 0; it < 16 && any; ++it) {
    any = false;
#pragma unroll
    for (int s = 0; s < NS; ++s) {
      const double ws = w[s];
      const double p = fma(fma(fma(fma(c4[s], ws, c3[s]), ws, c2[s]), ws, c1[s]), ws, c4[s]);
      const double dp = fma(fma(fma(4.0 * c4[s], ws, 3.0 * c3[s]), ws, 2.0 * c2[s]), ws, c1[s]);
      const double dw = p * dg_rcp_lo(dp);
      const double wn = ws - dw;
      const bool more = run[s] && !(fabs(dw) <= 1e-9 * wn);
      w[s] = run[s] ? wn : ws;
      run[s] = more;
      any = any || more;
    }
  }
#pragma unroll
  for (int s = 0; s < NS; ++s)
    if (general[s]) w[s] = dg_ideal_w_general(al, xi[s], eta[s]);
}

// Taub-Matthews: the positive root Wv = gamma^2 - 1 of the cubic of Eq. 61 with
// c1..c3 of Eq. 62-64.  The analytic route: Q, R, d of Eq. 65-67, the trigonometric branch Eq. 69-70
// (d < 0) or Cardano's Eq. 71-73 (d >= 0), with the safeguards of reading R7 (eta^2 - xi^2 =
// (eta-xi)(eta+xi), acos argument clamped, Wv >= 0).  The closed form returns Wv as a difference of
// O(c1) terms, so it is polished on the cubic itself by Newton steps (reading R7b), which makes the
// accuracy of the transcendental part irrelevant: it is evaluated in single precision and followed by
// two to four Newton steps with a convergence test on the last step (quadratic convergence from a
// 1e-7 seed).  A state that fails the test -- PAPER.md:392: Newton on this cubic "is not guaranteed to
// converge to the positive root" from a poor start -- takes the fallback: the same closed form in
// double precision plus two Newton steps; *nfall counts them.
// one Newton step on Eq. 61 with a single-precision reciprocal (self-correcting: the step's relative
// error 6e-8 only adds 6e-8 |dW| to the new iterate's error)
DG_INL double dg_tm_cubic_newton_lo(double Wv, double c1, double c2, double c3, double& dW) {
  const double f = fma(fma(Wv + c1, Wv, c2), Wv, c3);
  const double df = fma(fma(3.0, Wv, 2.0 * c1), Wv, c2);
  dW = -f * dg_rcp_lo(df);
  const double Wn = Wv + dW;
  return fmax(Wn, 0.0);
}
DG_INL double dg_tm_cubic_newton(double Wv, double c1, double c2, double c3, double& dW) {
  const double f = fma(fma(Wv + c1, Wv, c2), Wv, c3);
  const double df = fma(fma(3.0, Wv, 2.0 * c1), Wv, c2);
  const double Wn = Wv - f * dg_rcp(df);
  dW = Wn - Wv;
  return isfinite(Wn) ? fmax(Wn, 0.0) : Wv;
}

static __device__ __noinline__ double dg_tm_closed_form_fp64(double c1, double c2, double c3) {
  const double Q = (3.0 * c2 - c1 * c1) * (1.0 / 9.0);
  const double R = (9.0 * c1 * c2 - 27.0 * c3 - 2.0 * c1 * c1 * c1) * (1.0 / 54.0);
  const double Q3 = Q * Q * Q;
  const double d = fma(R, R, Q3);
  double Wv;
  if (d < 0.0) {
    const double arg = fmin(1.0, fmax(-1.0, R / sqrt(-Q3)));
    Wv = 2.0 * sqrt(-Q) * cos(acos(arg) * (1.0 / 3.0)) - c1 * (1.0 / 3.0);
  } else {
    const double sd = sqrt(d);
    Wv = cbrt(R + sd) + cbrt(R - sd) - c1 * (1.0 / 3.0);
  }
  Wv = fmax(Wv, 0.0);
  double dW;
  Wv = dg_tm_cubic_newton(Wv, c1, c2, c3, dW);
  Wv = dg_tm_cubic_newton(Wv, c1, c2, c3, dW);
  return Wv;
}

// Single-precision pieces of the closed form's starting point (their error only moves the seed):
// acos by the seven-term fit sqrt(1 - x) * poly(x) of Abramowitz & Stegun 4.4.46 (|err| <= 2e-8 on
// [0, 1], acos(-x) = pi - acos(x)); the real cube root by exp2(log2|x| / 3) on the SFU.
DG_INL float dg_acos_seed(float x) {
  const float ax = fabsf(x);
  float p = -0.0012624911f;
  p = fmaf(p, ax, 0.0066700901f);
  p = fmaf(p, ax, -0.0170881256f);
  p = fmaf(p, ax, 0.0308918810f);
  p = fmaf(p, ax, -0.0501743046f);
  p = fmaf(p, ax, 0.0889789874f);
  p = fmaf(p, ax, -0.2145988016f);
  p = fmaf(p, ax, 1.5707963050f);
  float sq;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(sq) : "f"(1.0f - ax));
  const float r = sq * p;
  return (x < 0.0f) ? 3.14159265f - r : r;
}
DG_INL float dg_cbrt_seed(float x) {
  return copysignf(exp2f(__log2f(fabsf(x)) * (1.0f / 3.0f)), x);
}

template <int NS>
DG_INL void dg_tm_solve_W(const double* D, const double* E, const double* Mabs, double* Wv, int* nfall) {
#pragma unroll
  for (int s = 0; s < NS; ++s) {
    const double rD = dg_rcp(D[s]);
    const double xi = Mabs[s] * rD, eta = E[s] * rD;                // Eq. 38
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
    double W0;
    if (d < 0.0) {
      const double rq = dg_rsqrt(-Q);                                        // 1/sqrt(-Q): serves both roots
      const float arg = fminf(1.0f, fmaxf(-1.0f, __double2float_rn(R * (rq * rq * rq))));
      const float th = dg_acos_seed(arg) * (1.0f / 3.0f);
      W0 = 2.0 * (-Q * rq) * (double)__cosf(th) - c1 * (1.0 / 3.0);          // Eq. 69-70 (th in [0, pi/3])
    } else {
      const double sd = dg_sqrt(d);
      const double p = R + sd, q = R - sd;
      const float pf = __double2float_rn(p), qf = __double2float_rn(q);
      double cs;
      if (fmaxf(fabsf(pf), fabsf(qf)) < 1e37f) cs = (double)(dg_cbrt_seed(pf) + dg_cbrt_seed(qf));
      else cs = cbrt(p) + cbrt(q);                                           // beyond the single-precision range
      W0 = cs - c1 * (1.0 / 3.0);                                            // Eq. 71-73
    }
    W0 = (W0 > 0.0) ? W0 : 0.0;                                              // (NaN -> 0 as well)
    // R7b polish: two steps square the ~1e-7 seed error twice; the step is a tight estimate of the error
    // before it, so |dW| <= 1e-9 W certifies the fp64 floor.  States that are not there yet (gamma -> 1,
    // where W is tiny against the seed's absolute error) take two more steps in full precision.
    double dW;
    W0 = dg_tm_cubic_newton_lo(W0, c1, c2, c3, dW);
    W0 = dg_tm_cubic_newton_lo(W0, c1, c2, c3, dW);
    if (!(fabs(dW) <= 1e-9 * W0)) {
      W0 = dg_tm_cubic_newton(W0, c1, c2, c3, dW);
      W0 = dg_tm_cubic_newton(W0, c1, c2, c3, dW);
      if (!(fabs(dW) <= fma(1e-13, W0, 1e-300))) {                           // not converged / NaN
        W0 = dg_tm_closed_form_fp64(c1, c2, c3);
        // overflowed coefficients (E/D beyond ~1e77) have no root to offer: fail the state (status 2)
        if (!isfinite(c1) || !isfinite(c2) || !isfinite(c3)) W0 = __longlong_as_double(0x7ff8000000000000LL);
        if (nfall) *nfall += 1;
      }
    }
    Wv[s] = W0;
  }
}

DG_INL bool dg_finite5(const double W[5]) {
  return isfinite(W[0]) && isfinite(W[1]) && isfinite(W[2]) && isfinite(W[3]) && isfinite(W[4]);
}

// con2prim of NS states in lockstep.  FULL: W[s] = [rho, u, P] (Eq. 55-57 / Eq. 74-75); else only the
// pressure P[s] (what the stage kernel keeps).  st[s]: status.  nfall (or NULL): += Taub-Matthews
// fallbacks.  Inputs failing Eq. 25 are rejected before either solver (status 1, outputs NaN);
// check = false: the caller has already established Eq. 25 for all NS states (the physicality
// operator's screen, which is stricter), so the test is skipped.
template <int EOS, int NS, bool FULL>
DG_INL void dg_con2prim_n(const EosPar& e, const double (*U)[5], double (*W)[5], double* P, int* st,
                          int* nfall, bool check = true, const double* Pguess = nullptr) {
  const double qnan = __longlong_as_double(0x7ff8000000000000LL);
  double D[NS], E[NS], Mabs[NS];
  bool adm[NS];
#pragma unroll
  for (int s = 0; s < NS; ++s) adm[s] = true;
  if (check) {
#pragma unroll
    for (int s = 0; s < NS; ++s) adm[s] = dg_admissible(U[s], 1.0);
  }
#pragma unroll
  for (int s = 0; s < NS; ++s) {
    // (an inadmissible state goes through the solver too -- every loop is bounded and nothing traps --
    // and its outputs are replaced by NaN below)
    D[s] = U[s][0];
    E[s] = U[s][4];
    Mabs[s] = dg_sqrt_p(fma(U[s][1], U[s][1], fma(U[s][2], U[s][2], U[s][3] * U[s][3])));
  }
  if (EOS == DG_EOS_IDEAL) {
    double w[NS];
    dg_ideal_solve_w<NS>(e, D, E, Mabs, Pguess, w);
#pragma unroll
    for (int s = 0; s < NS; ++s) {
      const double w2 = w[s] * w[s];
      const double op = 1.0 + w2, om = 1.0 - w2;
      const double r1 = dg_rcp(op);
      const double beta = 2.0 * w[s] * r1;                         // Eq. 58
      const double rho = D[s] * om * r1;                           // Eq. 55, 1/gamma = (1-w^2)/(1+w^2)
      const double Pv = (e.G - 1.0) * (E[s] - beta * Mabs[s] - rho);   // Eq. 57
      bool ok = (w[s] >= 0.0 && w[s] < 1.0) && isfinite(Pv) && (Pv > 0.0);
      if (FULL) {
        // u = gamma v = gamma beta M/|M|, gamma beta = 2w/(1-w^2)   (Eq. 56)
        const double sc = (Mabs[s] > 0.0) ? 2.0 * w[s] * dg_rcp(om * Mabs[s]) : 0.0;
        W[s][0] = rho; W[s][1] = sc * U[s][1]; W[s][2] = sc * U[s][2]; W[s][3] = sc * U[s][3]; W[s][4] = Pv;
        ok = ok && dg_finite5(W[s]);
      } else {
        P[s] = Pv;
      }
      st[s] = adm[s] ? (ok ? 0 : 2) : 1;
    }
  } else {
    double Wv[NS];
    dg_tm_solve_W<NS>(D, E, Mabs, Wv, nfall);
#pragma unroll
    for (int s = 0; s < NS; ++s) {
      const double g2 = Wv[s] + 1.0;
      const double rg = dg_rsqrt(g2);                              // 1/gamma, Eq. 74
      const double ug = dg_sqrt(Wv[s]);                            // gamma beta
      const double beta = ug * rg;
      const double rho = D[s] * rg;
      const double X = fma(-beta, Mabs[s], E[s]);                  // E - M.v
      const double X3 = 3.0 * X;
      const double rr = dg_rcp(FULL ? X3 * Mabs[s] : X3);          // one reciprocal for 1/(3X) and 1/|M|
      const double Pv = (X - rho) * (X + rho) * (FULL ? rr * Mabs[s] : rr);   // Eq. 75
      bool ok = isfinite(Pv) && (Pv > 0.0);
      if (FULL) {
        const double sc = ug * (rr * X3);                          // gamma beta / |M|
        W[s][0] = rho; W[s][1] = sc * U[s][1]; W[s][2] = sc * U[s][2]; W[s][3] = sc * U[s][3]; W[s][4] = Pv;
        ok = ok && dg_finite5(W[s]);
      } else {
        P[s] = Pv;
      }
      st[s] = adm[s] ? (ok ? 0 : 2) : 1;
    }
  }
#pragma unroll
  for (int s = 0; s < NS; ++s) {
    if (!adm[s]) {
      if (FULL) {
#pragma unroll
        for (int v = 0; v < 5; ++v) W[s][v] = qnan;
      } else {
        P[s] = qnan;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Physicality operator, per node (Eq. 28-37): largest s = s1 s2 in [0,1] such
// that Ubar + s (U_i - Ubar) is admissible.  Stage 2's root (Eq. 37) is evaluated in the
// cancellation-free form of reading R14 with the Minkowski form <A,B> = A_E B_E - A_D B_D - A_M.B_M
// and E -> (1-eps_q) E (R13c).
// ---------------------------------------------------------------------------------------------
// (out of line and by value: the rare path must not force the callers' node arrays into local memory)
struct DgState5 { double v[5]; };
static __device__ __noinline__ double dg_limiter_node_s(DgState5 Ubs, DgState5 Uis, double f /* 1-eps_q */) {
  const double* Ub = Ubs.v;
  const double* Ui = Uis.v;
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

// c2p_variant.cu -- the paper's comparison variants of con2prim (dgrhd_con2prim_batch_variant,
// DGRHD_C2P_ALTERNATE) in a translation unit of their own, compiled with -fmad=false.
//
// Why its own unit: Brent's method decides its next step by comparing rounded values, so two correct
// fp64 evaluations that round differently (nvcc contracts a*b+c into a fused multiply-add, the CPU oracle
// is built with -ffp-contract=off) walk different paths and the parity test could only assert an
// agreement fraction.  Without contraction, and with no explicit fma() in this file, every operation here is
// a correctly rounded IEEE operation (+, -, *, /, sqrt) in the order written, so the Taub-Matthews Brent
// solver can be compared with the oracle state by state.  (The analytic quartic also calls cos, acos and
// cbrt, whose CUDA and glibc versions differ in the last place: its test stays tolerance-based.)  These
// kernels exist to rerun the paper's section-3.3 comparison, not for the stage kernel, so the missing
// contraction costs nothing on the hot path.
#include "physics.cuh"

#define DG_VARIANT_NT 256

// ---------------------------------------------------------------------------------------------
// The paper's two comparison variants of con2prim ("four algorithms in all", the study of
// section 3.3).  Plain double precision, one state per call: they exist to rerun
// that comparison on B200 (dgrhd_con2prim_batch_variant), not for the stage kernel.
// ---------------------------------------------------------------------------------------------
// Ideal EOS, analytic route (:269-323, after Ryu et al. [15]): the physical root of
//   beta^4 + a3 beta^3 + a2 beta^2 + a1 beta + a0 = 0   (Eq. 39 with its beta^3 term restored, reading
// R17; a0..a3 of Eq. 40-43) by Ferrari's factorisation through the real root x of the resolvent cubic
// (Eq. 47-53: Eq. 48 reads 9 i1 i2; the T < 0 branch is 2 sqrt(-S) cos(acos(R/sqrt(-S^3))/3) - i1/3),
// B, C of Eq. 45-46, beta by Eq. 44, finishing Eq. 55-57.
DG_INL int dg_c2p_ideal_analytic(const EosPar& e, const double U[5], double W[5]) {
  const double D = U[0], E = U[4], G = e.G;
  const double Mabs = sqrt(U[1] * U[1] + U[2] * U[2] + U[3] * U[3]);
  const double xi = Mabs / D, eta = E / D;                                  // Eq. 38
  double beta = 0.0;
  if (xi > 0.0) {
    const double g1 = G - 1.0, den = g1 * g1 * (xi * xi + 1.0);
    const double a3 = -2.0 * G * g1 * xi * eta / den;                       // Eq. 40
    const double a2 = (G * G * eta * eta + 2.0 * g1 * xi * xi - g1 * g1) / den;   // Eq. 41
    const double a1 = -2.0 * G * xi * eta / den;                            // Eq. 42
    const double a0 = xi * xi / den;                                        // Eq. 43
    const double i1 = -a2, i2 = a3 * a1 - 4.0 * a0;                         // Eq. 51-52
    const double i3 = 4.0 * a2 * a0 - a1 * a1 - a3 * a3 * a0;               // Eq. 53
    const double R = (9.0 * i1 * i2 - 27.0 * i3 - 2.0 * i1 * i1 * i1) / 54.0;   // Eq. 48
    const double S = (3.0 * i2 - i1 * i1) / 9.0;                            // Eq. 49
    const double T = R * R + S * S * S;                                     // Eq. 50
    double x;
    if (T < 0.0) {                                                          // Eq. 47
      const double arg = fmin(1.0, fmax(-1.0, R / sqrt(-(S * S * S))));
      x = 2.0 * sqrt(-S) * cos(acos(arg) / 3.0) - i1 / 3.0;
    } else {
      const double sT = sqrt(T);
      x = cbrt(R + sT) + cbrt(R - sT) - i1 / 3.0;
    }
    const double B = 0.5 * (a3 + sqrt(a3 * a3 - 4.0 * a2 + 4.0 * x));       // Eq. 45
    const double C = 0.5 * (x - sqrt(x * x - 4.0 * a0));                    // Eq. 46
    beta = 0.5 * (-B + sqrt(B * B - 4.0 * C));                              // Eq. 44
  }
  const double ig = sqrt(1.0 - beta * beta);
  const double rho = D * ig;                                                // Eq. 55
  const double sc = (Mabs > 0.0) ? beta / (ig * Mabs) : 0.0;                // u = gamma beta M/|M|  (Eq. 56)
  W[0] = rho; W[1] = sc * U[1]; W[2] = sc * U[2]; W[3] = sc * U[3];
  W[4] = (G - 1.0) * (E - beta * Mabs - rho);                               // Eq. 57
  return ((beta >= 0.0 && beta < 1.0) && dg_finite5(W) && (W[4] > 0.0)) ? 0 : 2;
}

// Taub-Matthews, iterative route (:392): Brent's method [36] on the cubic of Eq. 61 in W = gamma^2 - 1,
// bracketed by gamma in [1, 200] and re-bracketed upwards while the root is not inside; at most
// max_iter iterations (the paper's Fig. 2 uses 25 and 50), stopped early when the bracket is 4 ulp.
DG_INL int dg_c2p_tm_brent(const double U[5], double Wp[5], int max_iter) {
  const double D = U[0], E = U[4];
  const double Mabs = sqrt(U[1] * U[1] + U[2] * U[2] + U[3] * U[3]);
  const double xi = Mabs / D, eta = E / D;
  const double x2 = xi * xi, e2 = eta * eta;
  const double dif = (eta - xi) * (eta + xi), den = dif * dif;
  const double sum = e2 + x2, br = 4.0 * sum - (x2 + 1.0);
  const double c1 = (sum * br - 14.0 * x2 * e2) / (2.0 * den);
  const double c2 = (br * br - 57.0 * x2 * e2) / (16.0 * den);
  const double c3 = -9.0 * x2 * e2 / (16.0 * den);
#define DG_TMF(W_) (((W_) + c1) * (W_) + c2) * (W_) + c3
  double a = 0.0, b = 200.0 * 200.0 - 1.0;
  double fa = c3, fb = DG_TMF(b);
  for (int k = 0; k < 40 && fb < 0.0; ++k) { b = 100.0 * (b + 1.0) - 1.0; fb = DG_TMF(b); }
  double Wv;
  if (fa == 0.0) Wv = a;
  else if (!(fa < 0.0 && fb >= 0.0)) Wv = __longlong_as_double(0x7ff8000000000000LL);
  else {
    double c = a, fc = fa, d = b - a, ee = d;
    for (int it = 0; it < max_iter; ++it) {
      if ((fb > 0.0 && fc > 0.0) || (fb < 0.0 && fc < 0.0)) { c = a; fc = fa; d = b - a; ee = d; }
      if (fabs(fc) < fabs(fb)) { a = b; b = c; c = a; fa = fb; fb = fc; fc = fa; }
      const double tol = 2.0 * 2.220446049250313e-16 * fabs(b), m = 0.5 * (c - b);
      if (fabs(m) <= tol || fb == 0.0) break;
      if (fabs(ee) >= tol && fabs(fa) > fabs(fb)) {
        double p, q;
        const double s = fb / fa;
        if (a == c) { p = 2.0 * m * s; q = 1.0 - s; }                        // secant
        else {                                                               // inverse quadratic
          const double qq = fa / fc, r = fb / fc;
          p = s * (2.0 * m * qq * (qq - r) - (b - a) * (r - 1.0));
          q = (qq - 1.0) * (r - 1.0) * (s - 1.0);
        }
        if (p > 0.0) q = -q; else p = -p;
        if (2.0 * p < fmin(3.0 * m * q - fabs(tol * q), fabs(ee * q))) { ee = d; d = p / q; }
        else { d = m; ee = m; }
      } else { d = m; ee = m; }
      a = b; fa = fb;
      b += (fabs(d) > tol) ? d : (m > 0.0 ? tol : -tol);
      fb = DG_TMF(b);
    }
    Wv = b;
  }
#undef DG_TMF
  Wv = fmax(Wv, 0.0) + 0.0 * Wv;                                            // clamp, keep NaN
  const double g = sqrt(Wv + 1.0), beta = sqrt(Wv / (Wv + 1.0));            // Eq. 74
  const double rho = D / g, ug = sqrt(Wv);
  const double X = E - beta * Mabs;
  const double sc = (Mabs > 0.0) ? ug / Mabs : 0.0;
  Wp[0] = rho; Wp[1] = sc * U[1]; Wp[2] = sc * U[2]; Wp[3] = sc * U[3];
  Wp[4] = (X - rho) * (X + rho) / (3.0 * X);                                // Eq. 75
  return (dg_finite5(Wp) && (Wp[4] > 0.0)) ? 0 : 2;
}


// one state per thread
template <int EOS>
__global__ void __launch_bounds__(DG_VARIANT_NT)
dg_c2p_variant_kernel(long long n, const double* __restrict__ U, double* __restrict__ W,
                      int* __restrict__ status, EosPar eos, int max_iter) {
  const long long i = (long long)blockIdx.x * DG_VARIANT_NT + threadIdx.x;
  if (i >= n) return;
  double u[5], w[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) u[v] = __ldg(U + v * n + i);
  int st = 1;
  if (dg_admissible(u, 1.0)) {
    st = (EOS == DG_EOS_IDEAL) ? dg_c2p_ideal_analytic(eos, u, w) : dg_c2p_tm_brent(u, w, max_iter);
  } else {
#pragma unroll
    for (int v = 0; v < 5; ++v) w[v] = __longlong_as_double(0x7ff8000000000000LL);
  }
#pragma unroll
  for (int v = 0; v < 5; ++v) W[v * n + i] = w[v];
  if (status) status[i] = st;
}

// launcher, declared in dgrhd.cu
cudaError_t dg_launch_c2p_variant(int eos, long long n, const double* U, double* W, int* status, EosPar e,
                                  int max_iter, cudaStream_t st) {
  const unsigned nb = (unsigned)((n + DG_VARIANT_NT - 1) / DG_VARIANT_NT);
  if (eos == DG_EOS_IDEAL) dg_c2p_variant_kernel<0><<<nb, DG_VARIANT_NT, 0, st>>>(n, U, W, status, e, max_iter);
  else dg_c2p_variant_kernel<1><<<nb, DG_VARIANT_NT, 0, st>>>(n, U, W, status, e, max_iter);
  return cudaGetLastError();
}

// basis.h -- host-side construction of the nodal operator tables of the CUDA path.
//
// Nodal Lagrange basis on tensor-product Gauss-Lobatto-Legendre points (Eq. 13-14;
// node family: DESIGN.md reading R1), N = p+1 points per direction, used as basis nodes and as
// quadrature points (collocation).  Built numerically here (Newton on the Legendre recurrence and
// barycentric differentiation), independently of the oracle's tables.
//   x[i]      nodes on [-1,1], ascending
//   w[i]      quadrature weights, sum = 2
//   Dhat[i][q] = w_q l_i'(x_q) / w_i   so that the volume term of Eq. 17 divided by the (diagonal)
//               mass matrix is   (2/h) sum_q Dhat[i][q] F(x_q)
//   lift      = 1/w_0 = 1/w_{N-1}: the surface term of Eq. 18 over the mass matrix is
//               (2/h) lift (delta_{i,0} Fhat_minus - delta_{i,N-1} Fhat_plus)
#pragma once
#include <cmath>

struct BasisTables {
  int N;
  double x[5], w[5];
  double Dhat[5][5];
  double lift;
};

namespace dgbasis {

// Legendre P_n(x) and derivative by the three-term recurrence.
inline void legendre(int n, double x, double& P, double& dP) {
  double p0 = 1.0, p1 = x;
  if (n == 0) { P = 1.0; dP = 0.0; return; }
  for (int k = 2; k <= n; ++k) {
    double pk = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / k;
    p0 = p1; p1 = pk;
  }
  P = p1;
  dP = (x * x == 1.0) ? 0.5 * n * (n + 1.0) * ((x > 0 || n % 2 == 1) ? 1.0 : -1.0)
                      : n * (p0 - x * p1) / (1.0 - x * x);
}

inline bool build(int N, BasisTables& T) {
  if (N < 1 || N > 5) return false;
  T.N = N;
  if (N == 1) {                       // p = 0: one node, midpoint rule, no derivative
    T.x[0] = 0.0; T.w[0] = 2.0; T.Dhat[0][0] = 0.0; T.lift = 0.5;
    return true;
  }
  const int n = N - 1;                // interior GLL nodes are the roots of P_n'
  const double pi = 3.14159265358979323846;
  T.x[0] = -1.0; T.x[n] = 1.0;
  for (int i = 1; i < n; ++i) {
    double xi = -std::cos(pi * i / n);            // Chebyshev-Lobatto start
    for (int it = 0; it < 100; ++it) {
      double P, dP;
      legendre(n, xi, P, dP);
      // P_n'' from the Legendre ODE: (1-x^2) P'' = 2x P' - n(n+1) P
      double d2P = (2.0 * xi * dP - n * (n + 1.0) * P) / (1.0 - xi * xi);
      double dx = dP / d2P;
      xi -= dx;
      if (std::fabs(dx) < 1e-16) break;
    }
    T.x[i] = xi;
  }
  for (int i = 0; i <= n / 2; ++i) {              // enforce exact symmetry
    double a = 0.5 * (T.x[n - i] - T.x[i]);
    T.x[i] = -a; T.x[n - i] = a;
  }
  for (int i = 0; i < N; ++i) {
    double P, dP;
    legendre(n, T.x[i], P, dP);
    T.w[i] = 2.0 / (n * (n + 1.0) * P * P);
  }
  // barycentric weights and the differentiation matrix Dm[q][i] = l_i'(x_q)
  double bw[5], Dm[5][5];
  for (int i = 0; i < N; ++i) {
    double p = 1.0;
    for (int k = 0; k < N; ++k) if (k != i) p *= (T.x[i] - T.x[k]);
    bw[i] = 1.0 / p;
  }
  for (int q = 0; q < N; ++q) {
    double diag = 0.0;
    for (int i = 0; i < N; ++i) {
      if (i == q) continue;
      Dm[q][i] = (bw[i] / bw[q]) / (T.x[q] - T.x[i]);
      diag -= Dm[q][i];
    }
    Dm[q][q] = diag;
  }
  for (int i = 0; i < N; ++i)
    for (int q = 0; q < N; ++q) T.Dhat[i][q] = T.w[q] * Dm[q][i] / T.w[i];
  T.lift = 1.0 / T.w[0];
  return true;
}

}  // namespace dgbasis

// hz_host_gll.h — host-side reference-element tables shared by the 2-D and 3-D drivers: GLL nodes, weights,
// differentiation matrix, K = D^T W D, Lambda_p, and the assembled 1-D band rows of a subdomain side.
#pragma once
#include <cmath>
#include <vector>

#include "hz_internal.h"

namespace hz {

// ------------------------------------------------------------------------------------------------
// GLL nodes, weights and differentiation matrix, from the Legendre recurrence.
// ------------------------------------------------------------------------------------------------
inline void legendre(int n, double x, double *Pn, double *dPn) {
  // P_n(x) and P_n'(x) by the three-term recurrence
  double p0 = 1.0, p1 = x, d0 = 0.0, d1 = 1.0;
  if (n == 0) { *Pn = 1.0; *dPn = 0.0; return; }
  for (int k = 2; k <= n; ++k) {
    const double p2 = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / k;
    const double d2 = d0 + (2.0 * k - 1.0) * p1;
    p0 = p1; p1 = p2; d0 = d1; d1 = d2;
  }
  *Pn = p1; *dPn = d1;
}

struct Gll {
  int p;
  double xi[kMaxP + 1], w[kMaxP + 1], D[kMaxP + 1][kMaxP + 1], K[kMaxP + 1][kMaxP + 1];
  double lambda_p;  // largest eigenvalue of the 1-D element pencil (K_h, W_h) at h = 1 (reading R9)
};

inline double sym_max_eig(int n, double A[kMaxP + 1][kMaxP + 1]) {
  // cyclic Jacobi on a small symmetric matrix
  double a[kMaxP + 1][kMaxP + 1];
  for (int i = 0; i < n; ++i) for (int j = 0; j < n; ++j) a[i][j] = A[i][j];
  for (int sweep = 0; sweep < 100; ++sweep) {
    double off = 0.0;
    for (int i = 0; i < n; ++i) for (int j = i + 1; j < n; ++j) off += a[i][j] * a[i][j];
    if (off < 1e-30) break;
    for (int pi = 0; pi < n; ++pi)
      for (int q = pi + 1; q < n; ++q) {
        if (std::fabs(a[pi][q]) < 1e-300) continue;
        const double th = (a[q][q] - a[pi][pi]) / (2.0 * a[pi][q]);
        const double t = (th >= 0 ? 1.0 : -1.0) / (std::fabs(th) + std::sqrt(th * th + 1.0));
        const double cs = 1.0 / std::sqrt(t * t + 1.0), sn = t * cs;
        for (int k = 0; k < n; ++k) {
          const double akp = a[k][pi], akq = a[k][q];
          a[k][pi] = cs * akp - sn * akq; a[k][q] = sn * akp + cs * akq;
        }
        for (int k = 0; k < n; ++k) {
          const double apk = a[pi][k], aqk = a[q][k];
          a[pi][k] = cs * apk - sn * aqk; a[q][k] = sn * apk + cs * aqk;
        }
      }
  }
  double mx = a[0][0];
  for (int i = 1; i < n; ++i) mx = std::fmax(mx, a[i][i]);
  return mx;
}

inline void make_gll(int p, Gll *g) {
  g->p = p;
  const int n = p + 1;
  g->xi[0] = -1.0; g->xi[p] = 1.0;
  // interior nodes: roots of P_p'(x); Chebyshev-Gauss-Lobatto initial guess + Newton with deflation-free
  // second derivative from the Legendre ODE: (1-x^2) P'' = 2x P' - p(p+1) P
  for (int a = 1; a < p; ++a) {
    double x = -std::cos(M_PI * a / p);
    for (int it = 0; it < 50; ++it) {
      double P, dP;
      legendre(p, x, &P, &dP);
      const double d2P = (2.0 * x * dP - p * (p + 1.0) * P) / (1.0 - x * x);
      const double dx = dP / d2P;
      x -= dx;
      if (std::fabs(dx) < 1e-16) break;
    }
    g->xi[a] = x;
  }
  if (p % 2 == 0) g->xi[p / 2] = 0.0;
  double Pv[kMaxP + 1];
  for (int a = 0; a < n; ++a) {
    double P, dP;
    legendre(p, g->xi[a], &P, &dP);
    Pv[a] = P;
    g->w[a] = 2.0 / (p * (p + 1.0) * P * P);
  }
  // D[a][b] = l_b'(xi_a) = P_p(xi_a) / (P_p(xi_b) (xi_a - xi_b)),  D[0][0] = -p(p+1)/4 = -D[p][p]
  for (int a = 0; a < n; ++a)
    for (int b = 0; b < n; ++b) {
      if (a != b) g->D[a][b] = Pv[a] / (Pv[b] * (g->xi[a] - g->xi[b]));
      else if (a == 0) g->D[a][b] = -0.25 * p * (p + 1.0);
      else if (a == p) g->D[a][b] = 0.25 * p * (p + 1.0);
      else g->D[a][b] = 0.0;
    }
  // K = D^T W D
  for (int a = 0; a < n; ++a)
    for (int b = 0; b < n; ++b) {
      double s = 0.0;
      for (int q = 0; q < n; ++q) s += g->D[q][a] * g->w[q] * g->D[q][b];
      g->K[a][b] = s;
    }
  // lambda_p = 4 * max eig(W^-1 K) = 4 * max eig(W^-1/2 K W^-1/2)
  double S[kMaxP + 1][kMaxP + 1];
  for (int a = 0; a < n; ++a)
    for (int b = 0; b < n; ++b) S[a][b] = g->K[a][b] / std::sqrt(g->w[a] * g->w[b]);
  g->lambda_p = 4.0 * sym_max_eig(n, S);
}

// Assembled 1-D operator rows of one subdomain side for the one-DOF-per-thread kernel:
// band[i][d] = (4/h^2) Kasm[i][i+d-P] / wasm[i], d = 0..2P (zero outside the side).
inline void make_band(const Gll &g, int ne, double h, std::vector<double> *band, std::vector<double> *wasm) {
  const int P = g.p, n = ne * P + 1, B = 2 * P + 1;
  std::vector<double> Kasm((size_t)n * B, 0.0);
  wasm->assign(n, 0.0);
  for (int e = 0; e < ne; ++e)
    for (int a = 0; a <= P; ++a) {
      (*wasm)[e * P + a] += g.w[a];
      for (int c = 0; c <= P; ++c) Kasm[(size_t)(e * P + a) * B + (c - a + P)] += g.K[a][c];
    }
  band->assign((size_t)n * B, 0.0);
  for (int i = 0; i < n; ++i)
    for (int d = 0; d < B; ++d) (*band)[(size_t)i * B + d] = 4.0 / (h * h) * Kasm[(size_t)i * B + d] / (*wasm)[i];
}


}  // namespace hz

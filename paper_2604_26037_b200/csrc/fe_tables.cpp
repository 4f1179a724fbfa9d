// fe_tables.cpp -- see fe_tables.h.  Host only, FP64.
#include "fe_tables.h"
#include <cmath>
#include <algorithm>

namespace pawfe {

void legendre(int n, double x, double* P, double* dP) {
  // (k+1) P_{k+1} = (2k+1) x P_k - k P_{k-1};  P_n' from  (1-x^2) P_n' = n (P_{n-1} - x P_n),
  // and the derivative recurrence P_{k+1}' = P_{k-1}' + (2k+1) P_k (valid at x = +-1 too).
  double p0 = 1.0, p1 = x, d0 = 0.0, d1 = 1.0;
  if (n == 0) { *P = 1.0; *dP = 0.0; return; }
  for (int k = 1; k < n; ++k) {
    double p2 = ((2 * k + 1) * x * p1 - k * p0) / (k + 1);
    double d2 = d0 + (2 * k + 1) * p1;
    p0 = p1; p1 = p2; d0 = d1; d1 = d2;
  }
  *P = p1; *dP = d1;
}

static double legendre_d2(int n, double x) {
  // (1-x^2) P'' - 2x P' + n(n+1) P = 0
  double P, dP;
  legendre(n, x, &P, &dP);
  return (2.0 * x * dP - n * (n + 1) * P) / (1.0 - x * x);
}

void gll_rule(int p, std::vector<double>& x, std::vector<double>& w) {
  const double pi = 3.14159265358979323846;
  x.assign(p + 1, 0.0); w.assign(p + 1, 0.0);
  x[0] = -1.0; x[p] = 1.0;
  for (int j = 1; j < p; ++j) {
    double t = -std::cos(pi * j / p);  // Chebyshev-Gauss-Lobatto guess
    for (int it = 0; it < 50; ++it) {
      double P, dP;
      legendre(p, t, &P, &dP);
      double dt = dP / legendre_d2(p, t);
      t -= dt;
      if (std::fabs(dt) < 1e-16) break;
    }
    x[j] = t;
  }
  // enforce exact antisymmetry
  for (int j = 0; j <= p / 2; ++j) { double a = 0.5 * (x[p - j] - x[j]); x[j] = -a; x[p - j] = a; }
  if (p % 2 == 0) x[p / 2] = 0.0;
  for (int j = 0; j <= p; ++j) {
    double P, dP;
    legendre(p, x[j], &P, &dP);
    w[j] = 2.0 / (p * (p + 1) * P * P);
  }
}

void gauss_legendre_rule(int n, std::vector<double>& x, std::vector<double>& w) {
  const double pi = 3.14159265358979323846;
  x.assign(n, 0.0); w.assign(n, 0.0);
  for (int i = 0; i < n; ++i) {
    double t = -std::cos(pi * (i + 0.75) / (n + 0.5));
    double P = 0, dP = 1;
    for (int it = 0; it < 100; ++it) {
      legendre(n, t, &P, &dP);
      double dt = P / dP;
      t -= dt;
      if (std::fabs(dt) < 1e-16) break;
    }
    legendre(n, t, &P, &dP);
    x[i] = t;
    w[i] = 2.0 / ((1.0 - t * t) * dP * dP);
  }
  for (int i = 0; i < n / 2; ++i) {
    double a = 0.5 * (x[n - 1 - i] - x[i]); x[i] = -a; x[n - 1 - i] = a;
    double ww = 0.5 * (w[i] + w[n - 1 - i]); w[i] = ww; w[n - 1 - i] = ww;
  }
  if (n % 2) x[n / 2] = 0.0;
}

void lagrange_basis(const std::vector<double>& nodes, const std::vector<double>& x,
                    std::vector<double>& L, std::vector<double>& dL) {
  int n = (int)nodes.size(), nx = (int)x.size();
  L.assign((size_t)n * nx, 0.0); dL.assign((size_t)n * nx, 0.0);
  for (int a = 0; a < n; ++a) {
    double den = 1.0;
    for (int b = 0; b < n; ++b) if (b != a) den *= (nodes[a] - nodes[b]);
    for (int i = 0; i < nx; ++i) {
      double num = 1.0;
      for (int b = 0; b < n; ++b) if (b != a) num *= (x[i] - nodes[b]);
      L[(size_t)a * nx + i] = num / den;
      double s = 0.0;
      for (int c = 0; c < n; ++c) {
        if (c == a) continue;
        double t = 1.0;
        for (int b = 0; b < n; ++b) if (b != a && b != c) t *= (x[i] - nodes[b]);
        s += t;
      }
      dL[(size_t)a * nx + i] = s / den;
    }
  }
}

void matrices_1d(int p, std::vector<double>& K1, std::vector<double>& M1, std::vector<double>& G1) {
  std::vector<double> xi, wg, xq, wq, L, dL;
  gll_rule(p, xi, wg);
  gauss_legendre_rule(p + 2, xq, wq);
  lagrange_basis(xi, xq, L, dL);
  int n1 = p + 1, nq = p + 2;
  K1.assign(n1 * n1, 0.0); M1.assign(n1 * n1, 0.0); G1.assign(n1 * n1, 0.0);
  for (int a = 0; a < n1; ++a)
    for (int b = 0; b < n1; ++b) {
      double k = 0, m = 0, g = 0;
      for (int q = 0; q < nq; ++q) {
        k += wq[q] * dL[a * nq + q] * dL[b * nq + q];
        m += wq[q] * L[a * nq + q] * L[b * nq + q];
        g += wq[q] * L[a * nq + q] * dL[b * nq + q];
      }
      K1[a * n1 + b] = k; M1[a * n1 + b] = m; G1[a * n1 + b] = g;
    }
}

void kron3(int n1, const std::vector<double>& A, const std::vector<double>& B,
           const std::vector<double>& C, double scale, std::vector<double>& out) {
  int n = n1 * n1 * n1;
  for (int a = 0; a < n1; ++a) for (int b = 0; b < n1; ++b) for (int c = 0; c < n1; ++c) {
    int I = (a * n1 + b) * n1 + c;
    for (int a2 = 0; a2 < n1; ++a2) {
      double va = scale * A[a * n1 + a2];
      for (int b2 = 0; b2 < n1; ++b2) {
        double vb = va * B[b * n1 + b2];
        for (int c2 = 0; c2 < n1; ++c2) {
          int J = (a2 * n1 + b2) * n1 + c2;
          out[(size_t)I * n + J] += vb * C[c * n1 + c2];
        }
      }
    }
  }
}

static inline void cmul(double ar, double ai, double br, double bi, double* r, double* i) {
  *r = ar * br - ai * bi; *i = ar * bi + ai * br;
}

bool solve_complex(int n, std::vector<double> A, std::vector<double> Bm, std::vector<double>& X) {
  // A, Bm: n x n complex interleaved.  Forward elimination with partial pivoting, back substitution.
  for (int k = 0; k < n; ++k) {
    int piv = k; double best = -1;
    for (int r = k; r < n; ++r) {
      double m = std::hypot(A[2 * (r * n + k)], A[2 * (r * n + k) + 1]);
      if (m > best) { best = m; piv = r; }
    }
    if (best <= 0) return false;
    if (piv != k)
      for (int c = 0; c < 2 * n; ++c) { std::swap(A[2 * k * n + c], A[2 * piv * n + c]); std::swap(Bm[2 * k * n + c], Bm[2 * piv * n + c]); }
    double pr = A[2 * (k * n + k)], pi_ = A[2 * (k * n + k) + 1], d = pr * pr + pi_ * pi_;
    double ir = pr / d, ii = -pi_ / d;
    for (int r = k + 1; r < n; ++r) {
      double fr, fi;
      cmul(A[2 * (r * n + k)], A[2 * (r * n + k) + 1], ir, ii, &fr, &fi);
      if (fr == 0 && fi == 0) continue;
      for (int c = k; c < n; ++c) {
        double tr, ti; cmul(fr, fi, A[2 * (k * n + c)], A[2 * (k * n + c) + 1], &tr, &ti);
        A[2 * (r * n + c)] -= tr; A[2 * (r * n + c) + 1] -= ti;
      }
      for (int c = 0; c < n; ++c) {
        double tr, ti; cmul(fr, fi, Bm[2 * (k * n + c)], Bm[2 * (k * n + c) + 1], &tr, &ti);
        Bm[2 * (r * n + c)] -= tr; Bm[2 * (r * n + c) + 1] -= ti;
      }
    }
  }
  X.assign((size_t)2 * n * n, 0.0);
  for (int c = 0; c < n; ++c)
    for (int r = n - 1; r >= 0; --r) {
      double sr = Bm[2 * (r * n + c)], si = Bm[2 * (r * n + c) + 1];
      for (int k = r + 1; k < n; ++k) {
        double tr, ti; cmul(A[2 * (r * n + k)], A[2 * (r * n + k) + 1], X[2 * (k * n + c)], X[2 * (k * n + c) + 1], &tr, &ti);
        sr -= tr; si -= ti;
      }
      double pr = A[2 * (r * n + r)], pi_ = A[2 * (r * n + r) + 1], d = pr * pr + pi_ * pi_;
      X[2 * (r * n + c)] = (sr * pr + si * pi_) / d;
      X[2 * (r * n + c) + 1] = (si * pr - sr * pi_) / d;
    }
  return true;
}

}  // namespace pawfe

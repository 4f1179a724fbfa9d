// fe_tables.h -- host-side 1-D spectral-element tables (GLL / Gauss-Legendre rules, Lagrange basis,
// reference-interval matrices).  PAPER.md:L116 (GLL nodal basis), L307 (tensor product), L321 (rules).
#pragma once
#include <vector>

namespace pawfe {

// Legendre P_n(x) and P_n'(x) by the three-term recurrence.
void legendre(int n, double x, double* P, double* dP);

// p+1 Gauss-Lobatto-Legendre nodes (ascending) and weights w = 2 / (p (p+1) P_p(x)^2).
void gll_rule(int p, std::vector<double>& x, std::vector<double>& w);

// n-point Gauss-Legendre rule on [-1, 1] (ascending nodes).
void gauss_legendre_rule(int n, std::vector<double>& x, std::vector<double>& w);

// L[a*nx + i] = l_a(x_i), dL likewise: Lagrange basis on `nodes` and its derivative at points x.
void lagrange_basis(const std::vector<double>& nodes, const std::vector<double>& x,
                    std::vector<double>& L, std::vector<double>& dL);

// K1 = int l_a' l_b', M1 = int l_a l_b, G1 = int l_a l_b'  on [-1,1], each (p+1)^2 row-major,
// integrated exactly with p+2 Gauss-Legendre points.
void matrices_1d(int p, std::vector<double>& K1, std::vector<double>& M1, std::vector<double>& G1);

// Kronecker product of three n1 x n1 matrices, order (x, y, z): out[(a*n1+b)*n1+c][(a'*n1+b')*n1+c']
void kron3(int n1, const std::vector<double>& A, const std::vector<double>& B,
           const std::vector<double>& C, double scale, std::vector<double>& out_accum);

// Solve A X = Bm for complex (or real with zero imaginary part) n x n, row-major interleaved
// (re, im); Gaussian elimination with partial pivoting.  Returns false if singular.
bool solve_complex(int n, std::vector<double> A, std::vector<double> Bm, std::vector<double>& X);

}  // namespace pawfe

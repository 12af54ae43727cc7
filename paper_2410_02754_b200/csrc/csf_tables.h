// csf_tables.h — host-side operator tables of the CUDA path (closed forms; independent of oracle/).
//
// 1-D GLL reference data on [-1,1] for the tensor-product Lagrange basis of degree p:
//   nodes xi_i = {+-1} U roots of P_p'  (found as eigenvalues of the Jacobi(1,1) tridiagonal matrix),
//   weights w_i = 2 / (p (p+1) P_p(xi_i)^2),
//   differentiation matrix D_qi = l_i'(xi_q) in closed form,
//   stiffness Khat = D^T diag(w) D   (exact: integrand degree 2p-2),
//   mass      Mhat = diag(w) - alpha v v^T,  v_i = w_i P_p(xi_i),  alpha = p(p+1)/(2(2p+1))   (exact).
// Per mesh direction d (cell size h, GLL-lumped 1-D mass m_i = (h/2) w_i, doubled on shared end nodes) the
// Loewdin-scaled 1-D operators used by the cell kernel are
//   A = 1/2 * s (2/h) Khat s,     B = s (h/2) Mhat s = diag(beta) - u u^T,   s_i = m_i^{-1/2},
// so that  S^(e) [1/2 K^(e)] S^(e) = Bz(x)By(x)Ax + Bz(x)Ay(x)Bx + Az(x)By(x)Bx   (eq.40 first term, eq.77).
#pragma once
#include <cstdint>
#include <vector>

namespace csf {

constexpr int kMaxN = 8;   // p <= 7

struct Gll1D {
    int p = 0, n = 0;
    double xi[kMaxN], w[kMaxN], v[kMaxN], alpha = 0.0;
    double K[kMaxN][kMaxN];   // Khat
    double D[kMaxN][kMaxN];   // D_qi = l_i'(xi_q); w_q D_qi = int l_q l_i' exactly (degree 2p - 1), the 1-D gradient matrix of eq.40's -i k.grad term
};

struct Dir1D {                // scaled 1-D operators of one mesh direction
    double A[kMaxN][kMaxN];   // 1/2 s (2/h) Khat s
    double beta[kMaxN];       // diagonal of B
    double u[kMaxN];          // rank-one part of B
    double m1d[kMaxN];        // lumped 1-D mass of the cell-local node (shared end nodes doubled)
};

bool build_gll(int p, Gll1D* g);
void build_dir(const Gll1D& g, double h, Dir1D* d);

// Gauss-Legendre rule with nq points on [-1,1] (eq.44): x ascending = zeros of P_nq (Newton from the
// Chebyshev guess), w = 2 / ((1 - x^2) P_nq'(x)^2). nq <= kMaxQ.
constexpr int kMaxQ = 16;
bool build_gauss_legendre(int nq, double* x, double* w);
// L[i * nq + q] = l_i(x[q]): the Lagrange polynomials on the GLL nodes of g at nq arbitrary points (eq.82, one direction)
void lagrange_at_points(const Gll1D& g, int nq, const double* x, double* L);

}  // namespace csf

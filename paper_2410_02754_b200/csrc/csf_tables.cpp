// csf_tables.cpp — closed-form GLL tables for the CUDA path (see csf_tables.h).
#include "csf_tables.h"

#include <algorithm>
#include <cmath>

namespace csf {

// P_p(x) and P_p'(x) through (k+1) P_{k+1} = (2k+1) x P_k - k P_{k-1} and
// (1-x^2) P_p' = p (P_{p-1} - x P_p); the end points use P_p'(+-1) = (+-1)^{p-1} p(p+1)/2.
static void legendre_pd(int p, double x, double* P, double* dP) {
    double pm = 1.0, pc = x;
    if (p == 0) { *P = 1.0; *dP = 0.0; return; }
    for (int k = 1; k < p; ++k) { double pn = ((2.0 * k + 1.0) * x * pc - k * pm) / (k + 1.0); pm = pc; pc = pn; }
    *P = pc;
    double om = 1.0 - x * x;
    if (om > 1e-12) *dP = p * (pm - x * pc) / om;
    else *dP = 0.5 * p * (p + 1.0) * ((x > 0 || (p % 2)) ? 1.0 : -1.0);
}

// eigenvalues of a small symmetric matrix by cyclic Jacobi rotations
static void jacobi_eigs(int n, double a[kMaxN][kMaxN], double* ev) {
    for (int sweep = 0; sweep < 60; ++sweep) {
        double off = 0.0;
        for (int i = 0; i < n; ++i) for (int j = i + 1; j < n; ++j) off += a[i][j] * a[i][j];
        if (off < 1e-32) break;
        for (int pi = 0; pi < n; ++pi) for (int q = pi + 1; q < n; ++q) {
            if (std::fabs(a[pi][q]) < 1e-300) continue;
            double th = (a[q][q] - a[pi][pi]) / (2.0 * a[pi][q]);
            double t = (th >= 0 ? 1.0 : -1.0) / (std::fabs(th) + std::sqrt(th * th + 1.0));
            double c = 1.0 / std::sqrt(t * t + 1.0), s = t * c;
            for (int k = 0; k < n; ++k) { double akp = a[k][pi], akq = a[k][q]; a[k][pi] = c * akp - s * akq; a[k][q] = s * akp + c * akq; }
            for (int k = 0; k < n; ++k) { double apk = a[pi][k], aqk = a[q][k]; a[pi][k] = c * apk - s * aqk; a[q][k] = s * apk + c * aqk; }
        }
    }
    for (int i = 0; i < n; ++i) ev[i] = a[i][i];
    std::sort(ev, ev + n);
}

bool build_gll(int p, Gll1D* g) {
    if (p < 1 || p + 1 > kMaxN) return false;
    const int n = p + 1;
    g->p = p; g->n = n;
    g->xi[0] = -1.0; g->xi[p] = 1.0;
    if (p >= 2) {
        // interior nodes = zeros of the Jacobi polynomial P^{(1,1)}_{p-1} = eigenvalues of the symmetric
        // tridiagonal matrix with zero diagonal and off-diagonal sqrt(k(k+2)/((2k+1)(2k+3))), k = 1..p-2
        double J[kMaxN][kMaxN] = {};
        for (int k = 1; k <= p - 2; ++k) { double b = std::sqrt(k * (k + 2.0) / ((2.0 * k + 1.0) * (2.0 * k + 3.0))); J[k - 1][k] = b; J[k][k - 1] = b; }
        double ev[kMaxN];
        jacobi_eigs(p - 1, J, ev);
        for (int i = 1; i < p; ++i) {
            double x = ev[i - 1];
            for (int it = 0; it < 4; ++it) {   // polish on q(x) = P_p'(x), q' from the Legendre ODE
                double P, dP; legendre_pd(p, x, &P, &dP);
                double ddP = (2.0 * x * dP - p * (p + 1.0) * P) / (1.0 - x * x);
                x -= dP / ddP;
            }
            g->xi[i] = x;
        }
        for (int i = 0; i < n / 2; ++i) { double a = 0.5 * (g->xi[n - 1 - i] - g->xi[i]); g->xi[i] = -a; g->xi[n - 1 - i] = a; }
        if (n % 2) g->xi[n / 2] = 0.0;
    }
    double Lp[kMaxN];
    for (int i = 0; i < n; ++i) { double P, dP; legendre_pd(p, g->xi[i], &P, &dP); Lp[i] = P; g->w[i] = 2.0 / (p * (p + 1.0) * P * P); g->v[i] = g->w[i] * P; }
    g->alpha = p * (p + 1.0) / (2.0 * (2.0 * p + 1.0));
    double D[kMaxN][kMaxN];
    for (int q = 0; q < n; ++q) for (int i = 0; i < n; ++i) D[q][i] = (q == i) ? 0.0 : Lp[q] / (Lp[i] * (g->xi[q] - g->xi[i]));
    D[0][0] = -0.25 * p * (p + 1.0); D[p][p] = 0.25 * p * (p + 1.0);
    for (int q = 0; q < n; ++q) for (int i = 0; i < n; ++i) g->D[q][i] = D[q][i];
    for (int i = 0; i < n; ++i) for (int j = 0; j < n; ++j) {
        double s = 0.0;
        for (int q = 0; q < n; ++q) s += D[q][i] * g->w[q] * D[q][j];
        g->K[i][j] = s;
    }
    return true;
}

void build_dir(const Gll1D& g, double h, Dir1D* d) {
    const int n = g.n, p = g.p;
    double s[kMaxN];
    for (int i = 0; i < n; ++i) {
        const bool shared = (i == 0 || i == p);
        d->m1d[i] = 0.5 * h * g.w[i] * (shared ? 2.0 : 1.0);
        s[i] = 1.0 / std::sqrt(d->m1d[i]);
        d->beta[i] = shared ? 0.5 : 1.0;
        d->u[i] = std::sqrt(g.alpha * 0.5 * h) * s[i] * g.v[i];
    }
    for (int i = 0; i < n; ++i) for (int j = 0; j < n; ++j) d->A[i][j] = 0.5 * s[i] * (2.0 / h) * g.K[i][j] * s[j];
}

bool build_gauss_legendre(int nq, double* x, double* w) {
    if (nq < 1 || nq > kMaxQ) return false;
    const double pi = 3.14159265358979323846;
    for (int i = 0; i < nq; ++i) {
        double t = -std::cos(pi * (i + 0.75) / (nq + 0.5)), P = 0.0, dP = 1.0;
        for (int it = 0; it < 100; ++it) {
            legendre_pd(nq, t, &P, &dP);
            const double dt = P / dP;
            t -= dt;
            if (std::fabs(dt) < 1e-16) break;
        }
        legendre_pd(nq, t, &P, &dP);
        x[i] = t; w[i] = 2.0 / ((1.0 - t * t) * dP * dP);
    }
    for (int i = 0; i < nq / 2; ++i) {             // exact symmetry
        const double a = 0.5 * (x[nq - 1 - i] - x[i]), ww = 0.5 * (w[i] + w[nq - 1 - i]);
        x[i] = -a; x[nq - 1 - i] = a; w[i] = ww; w[nq - 1 - i] = ww;
    }
    if (nq % 2) x[nq / 2] = 0.0;
    return true;
}

void lagrange_at_points(const Gll1D& g, int nq, const double* x, double* L) {
    for (int i = 0; i < g.n; ++i)
        for (int q = 0; q < nq; ++q) {
            double v = 1.0;
            for (int j = 0; j < g.n; ++j) if (j != i) v *= (x[q] - g.xi[j]) / (g.xi[i] - g.xi[j]);
            L[i * nq + q] = v;
        }
}

}  // namespace csf

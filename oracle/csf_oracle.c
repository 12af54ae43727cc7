/*
 * csf_oracle.c — the ORACLE. Plain, slow, obviously-correct CPU statement of
 *     Y = T_m(H~) X,  H~ = (Hhat - c I)/e,  Hhat = M_D^{-1/2} H M_D^{-1/2}
 * for the FE-discretised two-component spinor Hamiltonian of arxiv 2410.02754.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT. Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it. It shares no code,
 * header, table or constant generator with the CUDA path (paper_2410_02754_b200/csrc).
 *
 * What it follows (P:<line> = /root/reference/PAPER.md line, plus equation):
 *   - spinor coefficient layout U_{2I+alpha,n}                      P:300-302 (eq.38-39)
 *   - FE basis: tensor products of 1-D Lagrange polynomials of
 *     degree p on Gauss-Lobatto-Legendre nodes
 *   - integrals cell by cell with tensor Gauss-Legendre quadrature,
 *     weight w_q J^(e)                                             P:320-324 (eq.44)
 *   - H^loc: 1/2 grad N_I . grad N_J delta_ab + V_eff N_I N_J delta_ab
 *            + sum_d B^d N_I N_J sigma^d_ab  (k = 0)               P:304 (eq.40), P:523 (eq.77)
 *   - H^nloc = sum_a Pbar^a Delta^{gamma_a} Pbar^{a dagger},
 *     Delta_{2X+a,2X'+b} = D^{X X'}_{ab}                           P:308 (eq.41), P:517-519 (eq.76)
 *   - H = sum_e R^(e)T H^(e) R^(e) (assembly through the Boolean
 *     restriction matrices)                                        P:507 (eq.74)
 *   - M diagonal by GLL quadrature (M_D)                            P:461, P:317 (eq.43)
 *   - Chebyshev three-term recurrence                              P:465-467 (eq.70)
 * Readings taken where the paper is silent/garbled:
 *   A1 symmetric scaling M_D^{-1/2} H M_D^{-1/2}; A2 plain T_m; A3 stiffness integrated
 *   exactly (Gauss-Legendre, p+2 points); A4 V_eff,B collocated at the GLL nodes (mass-lumped
 *   potential block m_I (V_I I + B_I.sigma)); A5 P_{I chi} supplied already integrated;
 *   A6 eq.41 index order; A13 Dirichlet nodes removed.
 *
 * No blocking, fusion or reordering: the cell matrix is the literal 3-D quadrature sum,
 * H is assembled SPARSE (CSR, real M x M, shared by both spins) and applied row by row.
 * Parity pins: tests/test_oracle_pins.py (closed forms, invariants, brute force); every
 * exported routine here is pinned there; none is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { double re, im; } ref_c128;

enum { REF_OK = 0, REF_EINVAL = -1, REF_ENOMEM = -2, REF_ESTATE = -4 };
enum { REF_BC_PERIODIC = 0, REF_BC_DIRICHLET = 1, REF_BC_FREE = 2 };

#define MAXP 9
#define MAXN (MAXP + 1)
#define MAXQ (MAXP + 3)

typedef struct ref_ctx {
    int ncell[3], bc[3], p, n, n3;
    double box[3], h[3];
    int64_t nfull[3];   /* nodes per direction incl. constrained ones */
    int64_t nfree[3];   /* unconstrained nodes per direction */
    int64_t M;          /* unconstrained nodes per spin */
    int64_t E;          /* number of cells */
    double xi[MAXN], w[MAXN];            /* GLL nodes / weights on [-1,1] */
    int64_t *conn;      /* [E][n3] global node id or -1 (constrained) : the restriction R^(e) */
    double *mass;       /* [M] lumped mass m_I */
    double *Ke;         /* [n3][n3] cell matrix 1/2 K^(e) (all cells congruent: uniform mesh) */
    /* CSR of the assembled real M x M matrix 1/2 K */
    int64_t *rowptr; int32_t *col; double *val;
    /* nodal potential */
    int have_pot; double *veff; double *bxyz;
    /* projectors */
    int natoms; int64_t *node_ptr; int64_t *node_idx; int *nproj; int64_t *pval_ptr; double *pvals;
    int *atom_type; int ntypes; ref_c128 *delta; int64_t *delta_ptr;
    int *atom_distinct; /* [natoms] 1 if the atom's support lists every node once (then its rows of Y can be updated in parallel) */
} ref_ctx;

/* ------------------------------------------------------------------ */
/* O1: 1-D reference operators on [-1,1]                                */
/* ------------------------------------------------------------------ */

/* Legendre polynomial P_k(x) and derivative by the Bonnet recurrence. */
static void legendre(int k, double x, double *P, double *dP) {
    double p0 = 1.0, p1 = x, d0 = 0.0, d1 = 1.0;
    if (k == 0) { *P = 1.0; *dP = 0.0; return; }
    for (int j = 2; j <= k; j++) {
        double p2 = ((2.0 * j - 1.0) * x * p1 - (j - 1.0) * p0) / j;
        double d2 = d0 + (2.0 * j - 1.0) * p1;     /* P'_j = P'_{j-2} + (2j-1) P_{j-1} */
        p0 = p1; p1 = p2; d0 = d1; d1 = d2;
    }
    *P = p1; *dP = d1;
}

/* GLL nodes: +-1 and the roots of P_p'(x); weights 2/(p(p+1) P_p(xi)^2).  ("GLL nodal points") */
int ref_gll(int p, double *nodes, double *weights) {
    if (p < 1 || p > MAXP) return REF_EINVAL;
    int n = p + 1;
    nodes[0] = -1.0; nodes[p] = 1.0;
    for (int i = 1; i < p; i++) {
        double x = -cos(M_PI * i / p);            /* Chebyshev-Gauss-Lobatto start */
        for (int it = 0; it < 100; it++) {
            /* Newton on q(x) = P_p'(x); q' from Legendre ODE: (1-x^2)P'' = 2xP' - p(p+1)P */
            double P, dP; legendre(p, x, &P, &dP);
            double ddP = (2.0 * x * dP - p * (p + 1.0) * P) / (1.0 - x * x);
            double dx = dP / ddP;
            x -= dx;
            if (fabs(dx) < 1e-16) break;
        }
        nodes[i] = x;
    }
    /* symmetrise */
    for (int i = 0; i < n / 2; i++) { double a = 0.5 * (nodes[n - 1 - i] - nodes[i]); nodes[i] = -a; nodes[n - 1 - i] = a; }
    if (n % 2) nodes[n / 2] = 0.0;
    for (int i = 0; i < n; i++) { double P, dP; legendre(p, nodes[i], &P, &dP); weights[i] = 2.0 / (p * (p + 1.0) * P * P); }
    return REF_OK;
}

/* Gauss-Legendre rule with nq points: roots of P_nq, weights 2/((1-x^2) P_nq'(x)^2). */
int ref_gauss_legendre(int nq, double *x, double *w) {
    if (nq < 1 || nq > MAXQ) return REF_EINVAL;
    for (int i = 0; i < nq; i++) {
        double z = -cos(M_PI * (i + 0.75) / (nq + 0.5));
        for (int it = 0; it < 100; it++) {
            double P, dP; legendre(nq, z, &P, &dP);
            double dz = P / dP; z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        double P, dP; legendre(nq, z, &P, &dP);
        x[i] = z; w[i] = 2.0 / ((1.0 - z * z) * dP * dP);
    }
    return REF_OK;
}

/* Lagrange basis l_i on the nodes xi[0..n-1], by the product formula. */
static double lagrange(int n, const double *xi, int i, double x) {
    double v = 1.0;
    for (int j = 0; j < n; j++) if (j != i) v *= (x - xi[j]) / (xi[i] - xi[j]);
    return v;
}
/* l_i'(x) = sum_{k != i} 1/(xi_i - xi_k) prod_{j != i,k} (x - xi_j)/(xi_i - xi_j). */
static double dlagrange(int n, const double *xi, int i, double x) {
    double s = 0.0;
    for (int k = 0; k < n; k++) {
        if (k == i) continue;
        double v = 1.0 / (xi[i] - xi[k]);
        for (int j = 0; j < n; j++) if (j != i && j != k) v *= (x - xi[j]) / (xi[i] - xi[j]);
        s += v;
    }
    return s;
}

/* 1-D reference matrices by Gauss-Legendre quadrature with p+2 points (exact: degree 2p <= 2(p+2)-1):
 *   Khat_ij = int l_i' l_j',  Mhat_ij = int l_i l_j,  D_qi = l_i'(xi_q).   All n x n row-major. */
int ref_ref1d(int p, double *Khat, double *Mhat, double *D) {
    if (p < 1 || p > MAXP) return REF_EINVAL;
    int n = p + 1, nq = p + 2;
    double xi[MAXN], w[MAXN], xq[MAXQ], wq[MAXQ];
    ref_gll(p, xi, w); ref_gauss_legendre(nq, xq, wq);
    for (int i = 0; i < n; i++) for (int j = 0; j < n; j++) {
        double k = 0.0, m = 0.0;
        for (int q = 0; q < nq; q++) {
            k += wq[q] * dlagrange(n, xi, i, xq[q]) * dlagrange(n, xi, j, xq[q]);
            m += wq[q] * lagrange(n, xi, i, xq[q]) * lagrange(n, xi, j, xq[q]);
        }
        if (Khat) Khat[i * n + j] = k;
        if (Mhat) Mhat[i * n + j] = m;
        if (D) D[i * n + j] = dlagrange(n, xi, j, xi[i]);
    }
    return REF_OK;
}

/* ------------------------------------------------------------------ */
/* O2: mesh and numbering                                              */
/* ------------------------------------------------------------------ */

/* full 1-D node index g in [0, nfull) -> unconstrained index or -1. */
static int64_t free_index(const ref_ctx *c, int d, int64_t g) {
    if (c->bc[d] == REF_BC_PERIODIC) return g % ((int64_t)c->ncell[d] * c->p);
    if (c->bc[d] == REF_BC_DIRICHLET) { if (g == 0 || g == (int64_t)c->ncell[d] * c->p) return -1; return g - 1; }
    return g; /* FREE: every node kept */
}

/* ------------------------------------------------------------------ */
/* O4: cell matrix 1/2 K^(e), literal 3-D quadrature of eq.40/77 first term with eq.44          */
/* ------------------------------------------------------------------ */
static int build_cell_matrix(ref_ctx *c) {
    int n = c->n, n3 = c->n3, nq = c->p + 2;
    double xq[MAXQ], wq[MAXQ];
    ref_gauss_legendre(nq, xq, wq);
    /* basis values and derivatives at the 1-D quadrature points */
    double L[MAXN][MAXQ], dL[MAXN][MAXQ];
    for (int i = 0; i < n; i++) for (int q = 0; q < nq; q++) { L[i][q] = lagrange(n, c->xi, i, xq[q]); dL[i][q] = dlagrange(n, c->xi, i, xq[q]); }
    c->Ke = (double *)calloc((size_t)n3 * n3, sizeof(double));
    if (!c->Ke) return REF_ENOMEM;
    /* affine map: x = x0 + h_x (xt+1)/2  =>  d/dx = (2/h_x) d/dxt, J = h_x h_y h_z / 8 */
    double J = c->h[0] * c->h[1] * c->h[2] / 8.0;
    double gx = 2.0 / c->h[0], gy = 2.0 / c->h[1], gz = 2.0 / c->h[2];
#pragma omp parallel for schedule(static)
    for (int I = 0; I < n3; I++) {
        int i1 = I % n, j1 = (I / n) % n, k1 = I / (n * n);
        for (int Jn = 0; Jn < n3; Jn++) {
            int i2 = Jn % n, j2 = (Jn / n) % n, k2 = Jn / (n * n);
            double s = 0.0;
            for (int qz = 0; qz < nq; qz++) for (int qy = 0; qy < nq; qy++) for (int qx = 0; qx < nq; qx++) {
                double wJ = wq[qx] * wq[qy] * wq[qz] * J;
                /* grad N_I = (gx l_i' l_j l_k, gy l_i l_j' l_k, gz l_i l_j l_k') */
                double aIx = gx * dL[i1][qx] * L[j1][qy] * L[k1][qz];
                double aIy = gy * L[i1][qx] * dL[j1][qy] * L[k1][qz];
                double aIz = gz * L[i1][qx] * L[j1][qy] * dL[k1][qz];
                double aJx = gx * dL[i2][qx] * L[j2][qy] * L[k2][qz];
                double aJy = gy * L[i2][qx] * dL[j2][qy] * L[k2][qz];
                double aJz = gz * L[i2][qx] * L[j2][qy] * dL[k2][qz];
                s += wJ * 0.5 * (aIx * aJx + aIy * aJy + aIz * aJz);
            }
            c->Ke[(size_t)I * n3 + Jn] = s;
        }
    }
    return REF_OK;
}

/* ------------------------------------------------------------------ */
/* CSR assembly  H = sum_e R^T H^(e) R   (eq.74)                        */
/* ------------------------------------------------------------------ */
static int cmp_i64(const void *a, const void *b) { int64_t x = *(const int64_t *)a, y = *(const int64_t *)b; return (x > y) - (x < y); }

static int assemble_csr(ref_ctx *c) {
    int n3 = c->n3; int64_t M = c->M, E = c->E;
    /* node -> cells incidence (each node belongs to at most 8 cells) */
    int *cnt = (int *)calloc((size_t)M, sizeof(int));
    int64_t *inc = (int64_t *)malloc((size_t)M * 8 * 2 * sizeof(int64_t)); /* (cell, local) pairs */
    if (!cnt || !inc) return REF_ENOMEM;
    for (int64_t e = 0; e < E; e++) for (int l = 0; l < n3; l++) {
        int64_t I = c->conn[e * n3 + l]; if (I < 0) continue;
        int k = cnt[I]++; if (k >= 8) return REF_EINVAL;
        inc[(I * 8 + k) * 2] = e; inc[(I * 8 + k) * 2 + 1] = l;
    }
    c->rowptr = (int64_t *)malloc((size_t)(M + 1) * sizeof(int64_t));
    if (!c->rowptr) return REF_ENOMEM;
    /* pass 1: count distinct columns per row */
    int64_t *rownnz = (int64_t *)malloc((size_t)M * sizeof(int64_t));
#pragma omp parallel
    {
        int64_t *tmp = (int64_t *)malloc((size_t)8 * n3 * sizeof(int64_t));
#pragma omp for schedule(static)
        for (int64_t I = 0; I < M; I++) {
            int m = 0;
            for (int k = 0; k < cnt[I]; k++) { int64_t e = inc[(I * 8 + k) * 2];
                for (int l = 0; l < n3; l++) { int64_t Jg = c->conn[e * n3 + l]; if (Jg >= 0) tmp[m++] = Jg; } }
            qsort(tmp, m, sizeof(int64_t), cmp_i64);
            int u = 0; for (int t = 0; t < m; t++) if (t == 0 || tmp[t] != tmp[t - 1]) u++;
            rownnz[I] = u;
        }
        free(tmp);
    }
    c->rowptr[0] = 0; for (int64_t I = 0; I < M; I++) c->rowptr[I + 1] = c->rowptr[I] + rownnz[I];
    int64_t nnz = c->rowptr[M];
    c->col = (int32_t *)malloc((size_t)nnz * sizeof(int32_t));
    c->val = (double *)calloc((size_t)nnz, sizeof(double));
    if (!c->col || !c->val) return REF_ENOMEM;
    /* pass 2: fill pattern and add the cell-matrix entries */
#pragma omp parallel
    {
        int64_t *tmp = (int64_t *)malloc((size_t)8 * n3 * sizeof(int64_t));
#pragma omp for schedule(static)
        for (int64_t I = 0; I < M; I++) {
            int m = 0;
            for (int k = 0; k < cnt[I]; k++) { int64_t e = inc[(I * 8 + k) * 2];
                for (int l = 0; l < n3; l++) { int64_t Jg = c->conn[e * n3 + l]; if (Jg >= 0) tmp[m++] = Jg; } }
            qsort(tmp, m, sizeof(int64_t), cmp_i64);
            int64_t base = c->rowptr[I]; int u = 0;
            for (int t = 0; t < m; t++) if (t == 0 || tmp[t] != tmp[t - 1]) c->col[base + u++] = (int32_t)tmp[t];
            for (int k = 0; k < cnt[I]; k++) {
                int64_t e = inc[(I * 8 + k) * 2]; int li = (int)inc[(I * 8 + k) * 2 + 1];
                for (int l = 0; l < n3; l++) {
                    int64_t Jg = c->conn[e * n3 + l]; if (Jg < 0) continue;
                    /* binary search the column */
                    int lo = 0, hi = u - 1, pos = -1;
                    while (lo <= hi) { int mid = (lo + hi) / 2; int32_t cv = c->col[base + mid]; if (cv == (int32_t)Jg) { pos = mid; break; } if (cv < (int32_t)Jg) lo = mid + 1; else hi = mid - 1; }
                    c->val[base + pos] += c->Ke[(size_t)li * n3 + l];
                }
            }
        }
        free(tmp);
    }
    free(rownnz); free(cnt); free(inc);
    return REF_OK;
}

/* ------------------------------------------------------------------ */
/* context                                                             */
/* ------------------------------------------------------------------ */
int ref_destroy(ref_ctx *c) {
    if (!c) return REF_OK;
    free(c->conn); free(c->mass); free(c->Ke); free(c->rowptr); free(c->col); free(c->val);
    free(c->veff); free(c->bxyz);
    free(c->node_ptr); free(c->node_idx); free(c->nproj); free(c->pval_ptr); free(c->pvals);
    free(c->atom_type); free(c->delta); free(c->delta_ptr); free(c->atom_distinct);
    free(c);
    return REF_OK;
}

/* assemble_sparse = 0 skips the global CSR (then only ref_apply_H_rows / metadata calls work). */
int ref_create2(ref_ctx **out, const int ncell[3], const double box[3], int order, const int bc[3], int assemble_sparse) {
    if (!out || !ncell || !box || !bc || order < 1 || order > MAXP) return REF_EINVAL;
    for (int d = 0; d < 3; d++) if (ncell[d] < 1 || !(box[d] > 0.0) || bc[d] < 0 || bc[d] > 2) return REF_EINVAL;
    ref_ctx *c = (ref_ctx *)calloc(1, sizeof(ref_ctx));
    if (!c) return REF_ENOMEM;
    c->p = order; c->n = order + 1; c->n3 = c->n * c->n * c->n;
    c->E = 1; c->M = 1;
    for (int d = 0; d < 3; d++) {
        c->ncell[d] = ncell[d]; c->box[d] = box[d]; c->bc[d] = bc[d]; c->h[d] = box[d] / ncell[d];
        c->nfull[d] = (int64_t)ncell[d] * order + 1;
        c->nfree[d] = bc[d] == REF_BC_PERIODIC ? (int64_t)ncell[d] * order : (bc[d] == REF_BC_DIRICHLET ? (int64_t)ncell[d] * order - 1 : (int64_t)ncell[d] * order + 1);
        if (c->nfree[d] < 1) { free(c); return REF_EINVAL; }
        /* a periodic direction with a single cell of order 1 would alias both cell nodes */
        c->E *= ncell[d]; c->M *= c->nfree[d];
    }
    ref_gll(order, c->xi, c->w);
    int n = c->n, n3 = c->n3;
    /* R^(e): local (i,j,k), x fastest -> global id gx + Nx (gy + Ny gz) over unconstrained nodes */
    c->conn = (int64_t *)malloc((size_t)c->E * n3 * sizeof(int64_t));
    c->mass = (double *)calloc((size_t)c->M, sizeof(double));
    if (!c->conn || !c->mass) { ref_destroy(c); return REF_ENOMEM; }
    double J = c->h[0] * c->h[1] * c->h[2] / 8.0;
    for (int64_t e = 0; e < c->E; e++) {
        int64_t cx = e % ncell[0], cy = (e / ncell[0]) % ncell[1], cz = e / ((int64_t)ncell[0] * ncell[1]);
        for (int k = 0; k < n; k++) for (int j = 0; j < n; j++) for (int i = 0; i < n; i++) {
            int64_t fx = free_index(c, 0, cx * order + i), fy = free_index(c, 1, cy * order + j), fz = free_index(c, 2, cz * order + k);
            int64_t I = (fx < 0 || fy < 0 || fz < 0) ? -1 : fx + c->nfree[0] * (fy + c->nfree[1] * fz);
            c->conn[e * n3 + i + n * (j + n * k)] = I;
            /* O3 lumped mass: GLL quadrature of int N_I N_J is diagonal, m_I = sum_e J w_i w_j w_k */
            if (I >= 0) c->mass[I] += J * c->w[i] * c->w[j] * c->w[k];
        }
    }
    int rc = build_cell_matrix(c);
    if (rc == REF_OK && assemble_sparse) rc = assemble_csr(c);
    if (rc != REF_OK) { ref_destroy(c); return rc; }
    *out = c;
    return REF_OK;
}
int ref_create(ref_ctx **out, const int ncell[3], const double box[3], int order, const int bc[3]) {
    return ref_create2(out, ncell, box, order, bc, 1);
}

int ref_num_nodes(const ref_ctx *c, int64_t *M) { if (!c || !M) return REF_EINVAL; *M = c->M; return REF_OK; }
int ref_num_cells(const ref_ctx *c, int64_t *E) { if (!c || !E) return REF_EINVAL; *E = c->E; return REF_OK; }

int ref_node_coords(const ref_ctx *c, double *xyz) {
    if (!c || !xyz) return REF_EINVAL;
    int n = c->n, n3 = c->n3;
    for (int64_t e = 0; e < c->E; e++) {
        int64_t cc[3] = { e % c->ncell[0], (e / c->ncell[0]) % c->ncell[1], e / ((int64_t)c->ncell[0] * c->ncell[1]) };
        for (int l = 0; l < n3; l++) {
            int64_t I = c->conn[e * n3 + l]; if (I < 0) continue;
            int loc[3] = { l % n, (l / n) % n, l / (n * n) };
            for (int d = 0; d < 3; d++) {
                double x = (cc[d] + 0.5 * (c->xi[loc[d]] + 1.0)) * c->h[d];
                /* a periodic node is reported once, at its image inside [0, box) */
                if (c->bc[d] == REF_BC_PERIODIC && cc[d] == c->ncell[d] - 1 && loc[d] == c->p) x = 0.0;
                xyz[I * 3 + d] = x;
            }
        }
    }
    return REF_OK;
}
int ref_mass_diag(const ref_ctx *c, double *m) { if (!c || !m) return REF_EINVAL; memcpy(m, c->mass, (size_t)c->M * sizeof(double)); return REF_OK; }
int ref_connectivity(const ref_ctx *c, int64_t *conn) { if (!c || !conn) return REF_EINVAL; memcpy(conn, c->conn, (size_t)c->E * c->n3 * sizeof(int64_t)); return REF_OK; }
int ref_cell_matrix(const ref_ctx *c, double *Ke) { if (!c || !Ke) return REF_EINVAL; memcpy(Ke, c->Ke, (size_t)c->n3 * c->n3 * sizeof(double)); return REF_OK; }
int ref_csr_nnz(const ref_ctx *c, int64_t *nnz) { if (!c || !nnz || !c->rowptr) return REF_ESTATE; *nnz = c->rowptr[c->M]; return REF_OK; }
int ref_csr(const ref_ctx *c, int64_t *rowptr, int32_t *col, double *val) {
    if (!c || !c->rowptr) return REF_ESTATE;
    memcpy(rowptr, c->rowptr, (size_t)(c->M + 1) * sizeof(int64_t));
    memcpy(col, c->col, (size_t)c->rowptr[c->M] * sizeof(int32_t));
    memcpy(val, c->val, (size_t)c->rowptr[c->M] * sizeof(double));
    return REF_OK;
}

/* O5: nodal potential values V_I, B_I (A4).  bxyz == NULL => B = 0. */
int ref_set_potential(ref_ctx *c, const double *veff, const double *bxyz) {
    if (!c || !veff) return REF_EINVAL;
    free(c->veff); free(c->bxyz);
    c->veff = (double *)malloc((size_t)c->M * sizeof(double));
    c->bxyz = (double *)calloc((size_t)c->M * 3, sizeof(double));
    if (!c->veff || !c->bxyz) return REF_ENOMEM;
    memcpy(c->veff, veff, (size_t)c->M * sizeof(double));
    if (bxyz) memcpy(c->bxyz, bxyz, (size_t)c->M * 3 * sizeof(double));
    c->have_pot = 1;
    return REF_OK;
}

/* O6: projectors P_{I chi} (integrated values, A5) on each atom's support rows, and Delta per type. */
int ref_set_projectors(ref_ctx *c, int natoms, const int64_t *node_ptr, const int64_t *node_idx, const int *nproj,
                       const double *pvals, const int *atom_type, int ntypes, const ref_c128 *delta, const int64_t *delta_ptr) {
    if (!c || natoms < 0) return REF_EINVAL;
    free(c->node_ptr); free(c->node_idx); free(c->nproj); free(c->pval_ptr); free(c->pvals);
    free(c->atom_type); free(c->delta); free(c->delta_ptr); free(c->atom_distinct); c->atom_distinct = NULL;
    c->node_ptr = NULL; c->node_idx = NULL; c->nproj = NULL; c->pval_ptr = NULL; c->pvals = NULL;
    c->atom_type = NULL; c->delta = NULL; c->delta_ptr = NULL; c->natoms = 0; c->ntypes = 0;
    if (natoms == 0) return REF_OK;
    if (!node_ptr || !node_idx || !nproj || !pvals || !atom_type || ntypes < 1 || !delta || !delta_ptr) return REF_EINVAL;
    for (int a = 0; a < natoms; a++) {
        if (atom_type[a] < 0 || atom_type[a] >= ntypes || nproj[a] < 1) return REF_EINVAL;
        int64_t dn = delta_ptr[atom_type[a] + 1] - delta_ptr[atom_type[a]];
        if (dn != (int64_t)4 * nproj[a] * nproj[a]) return REF_EINVAL;
        for (int64_t t = node_ptr[a]; t < node_ptr[a + 1]; t++) if (node_idx[t] < 0 || node_idx[t] >= c->M) return REF_EINVAL;
    }
    int64_t nn = node_ptr[natoms];
    c->node_ptr = (int64_t *)malloc((size_t)(natoms + 1) * sizeof(int64_t));
    c->node_idx = (int64_t *)malloc((size_t)(nn ? nn : 1) * sizeof(int64_t));
    c->nproj = (int *)malloc((size_t)natoms * sizeof(int));
    c->pval_ptr = (int64_t *)malloc((size_t)(natoms + 1) * sizeof(int64_t));
    c->atom_type = (int *)malloc((size_t)natoms * sizeof(int));
    c->delta_ptr = (int64_t *)malloc((size_t)(ntypes + 1) * sizeof(int64_t));
    memcpy(c->node_ptr, node_ptr, (size_t)(natoms + 1) * sizeof(int64_t));
    memcpy(c->node_idx, node_idx, (size_t)nn * sizeof(int64_t));
    memcpy(c->nproj, nproj, (size_t)natoms * sizeof(int));
    memcpy(c->atom_type, atom_type, (size_t)natoms * sizeof(int));
    memcpy(c->delta_ptr, delta_ptr, (size_t)(ntypes + 1) * sizeof(int64_t));
    c->pval_ptr[0] = 0;
    for (int a = 0; a < natoms; a++) c->pval_ptr[a + 1] = c->pval_ptr[a] + (node_ptr[a + 1] - node_ptr[a]) * nproj[a];
    c->pvals = (double *)malloc((size_t)(c->pval_ptr[natoms] ? c->pval_ptr[natoms] : 1) * sizeof(double));
    memcpy(c->pvals, pvals, (size_t)c->pval_ptr[natoms] * sizeof(double));
    c->delta = (ref_c128 *)malloc((size_t)delta_ptr[ntypes] * sizeof(ref_c128));
    memcpy(c->delta, delta, (size_t)delta_ptr[ntypes] * sizeof(ref_c128));
    c->atom_distinct = (int *)malloc((size_t)natoms * sizeof(int));
    for (int a = 0; a < natoms; a++) {
        int64_t na = node_ptr[a + 1] - node_ptr[a];
        int64_t *tmp = (int64_t *)malloc((size_t)(na ? na : 1) * sizeof(int64_t));
        memcpy(tmp, node_idx + node_ptr[a], (size_t)na * sizeof(int64_t));
        qsort(tmp, (size_t)na, sizeof(int64_t), cmp_i64);
        int ok = 1; for (int64_t t = 1; t < na; t++) if (tmp[t] == tmp[t - 1]) ok = 0;
        c->atom_distinct[a] = ok; free(tmp);
    }
    c->natoms = natoms; c->ntypes = ntypes;
    return REF_OK;
}

/* ------------------------------------------------------------------ */
/* O7: Y = S (H (S X)),  S = M_D^{-1/2},  H = H^loc + H^nloc            */
/* ------------------------------------------------------------------ */
static inline ref_c128 cmul(ref_c128 a, ref_c128 b) { ref_c128 r = { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re }; return r; }

/* element (node I, spin s, vector v) lives at [(2I+s)*ld + v]   (P:302 row index 2I+alpha) */
int ref_apply_H(ref_ctx *c, const ref_c128 *X, ref_c128 *Y, int64_t ld, int nvec) {
    if (!c || !X || !Y || nvec < 0 || ld < nvec) return REF_EINVAL;
    if (!c->have_pot || !c->rowptr) return REF_ESTATE;
    int64_t M = c->M;
    /* Z = S X */
    ref_c128 *Z = (ref_c128 *)malloc((size_t)2 * M * (nvec ? nvec : 1) * sizeof(ref_c128));
    if (!Z) return REF_ENOMEM;
#pragma omp parallel for schedule(static)
    for (int64_t I = 0; I < M; I++) {
        double s = 1.0 / sqrt(c->mass[I]);
        for (int a = 0; a < 2; a++) for (int v = 0; v < nvec; v++) {
            ref_c128 x = X[(2 * I + a) * ld + v];
            Z[(2 * I + a) * (int64_t)nvec + v].re = s * x.re; Z[(2 * I + a) * (int64_t)nvec + v].im = s * x.im;
        }
    }
    /* local part, row by row: kinetic CSR (identical for both spins, delta_ab) + lumped 2x2 potential block */
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t I = 0; I < M; I++) {
        for (int a = 0; a < 2; a++) for (int v = 0; v < nvec; v++) { Y[(2 * I + a) * ld + v].re = 0.0; Y[(2 * I + a) * ld + v].im = 0.0; }
        for (int64_t t = c->rowptr[I]; t < c->rowptr[I + 1]; t++) {
            int64_t Jn = c->col[t]; double k = c->val[t];
            for (int a = 0; a < 2; a++) {
                const ref_c128 *z = Z + (2 * Jn + a) * (int64_t)nvec; ref_c128 *y = Y + (2 * I + a) * ld;
                for (int v = 0; v < nvec; v++) { y[v].re += k * z[v].re; y[v].im += k * z[v].im; }
            }
        }
        /* m_I (V_I I + B_I . sigma): [[V+Bz, Bx - iBy],[Bx + iBy, V-Bz]]   (eq.16, eq.40; sigma from P:46) */
        double m = c->mass[I], V = c->veff[I], Bx = c->bxyz[3 * I], By = c->bxyz[3 * I + 1], Bz = c->bxyz[3 * I + 2];
        ref_c128 h00 = { m * (V + Bz), 0.0 }, h01 = { m * Bx, -m * By }, h10 = { m * Bx, m * By }, h11 = { m * (V - Bz), 0.0 };
        const ref_c128 *zu = Z + (2 * I) * (int64_t)nvec, *zd = Z + (2 * I + 1) * (int64_t)nvec;
        ref_c128 *yu = Y + (2 * I) * ld, *yd = Y + (2 * I + 1) * ld;
        for (int v = 0; v < nvec; v++) {
            ref_c128 t0 = cmul(h00, zu[v]), t1 = cmul(h01, zd[v]), t2 = cmul(h10, zu[v]), t3 = cmul(h11, zd[v]);
            yu[v].re += t0.re + t1.re; yu[v].im += t0.im + t1.im;
            yd[v].re += t2.re + t3.re; yd[v].im += t2.im + t3.im;
        }
    }
    /* nonlocal part, atom by atom: C = Pbar^dagger Z ; Ct = Delta C ; Y += Pbar Ct   (eq.41, eq.76; P real at k=0) */
    for (int a = 0; a < c->natoms; a++) {
        int np = c->nproj[a]; int64_t n0 = c->node_ptr[a], na = c->node_ptr[a + 1] - n0;
        const double *P = c->pvals + c->pval_ptr[a];
        const ref_c128 *D = c->delta + c->delta_ptr[c->atom_type[a]];
        size_t csz = (size_t)2 * np * (nvec ? nvec : 1);
        ref_c128 *C = (ref_c128 *)calloc(csz, sizeof(ref_c128)), *Ct = (ref_c128 *)calloc(csz, sizeof(ref_c128));
        /* C_{2X+s, v} = sum_I conj(P_{I X}) Z_{2I+s, v}.  (OpenMP over the projector index X: every C entry is still
         * summed over the support nodes t in the same order by one thread, so the arithmetic is unchanged.) */
#pragma omp parallel for schedule(static)
        for (int x = 0; x < np; x++) {
            for (int64_t t = 0; t < na; t++) { int64_t I = c->node_idx[n0 + t]; double pv = P[t * np + x];
                for (int s = 0; s < 2; s++) for (int v = 0; v < nvec; v++) {
                    C[(size_t)(2 * x + s) * nvec + v].re += pv * Z[(2 * I + s) * (int64_t)nvec + v].re;
                    C[(size_t)(2 * x + s) * nvec + v].im += pv * Z[(2 * I + s) * (int64_t)nvec + v].im; } } }
        /* Ct = Delta C */
        for (int r = 0; r < 2 * np; r++) for (int q = 0; q < 2 * np; q++) { ref_c128 d = D[(size_t)r * 2 * np + q];
            for (int v = 0; v < nvec; v++) { ref_c128 t = cmul(d, C[(size_t)q * nvec + v]); Ct[(size_t)r * nvec + v].re += t.re; Ct[(size_t)r * nvec + v].im += t.im; } }
        /* Y_{2I+s} += sum_X P_{I X} Ct_{2X+s}.  (OpenMP over the support nodes of this atom: they are distinct rows of Y,
         * and every row still adds its projector terms X in the same order.) */
#pragma omp parallel for schedule(static) if (c->atom_distinct[a])
        for (int64_t t = 0; t < na; t++) { int64_t I = c->node_idx[n0 + t];
            for (int x = 0; x < np; x++) { double pv = P[t * np + x];
                for (int s = 0; s < 2; s++) for (int v = 0; v < nvec; v++) {
                    Y[(2 * I + s) * ld + v].re += pv * Ct[(size_t)(2 * x + s) * nvec + v].re;
                    Y[(2 * I + s) * ld + v].im += pv * Ct[(size_t)(2 * x + s) * nvec + v].im; } } }
        free(C); free(Ct);
    }
    /* Y <- S Y */
#pragma omp parallel for schedule(static)
    for (int64_t I = 0; I < M; I++) {
        double s = 1.0 / sqrt(c->mass[I]);
        for (int a = 0; a < 2; a++) for (int v = 0; v < nvec; v++) { Y[(2 * I + a) * ld + v].re *= s; Y[(2 * I + a) * ld + v].im *= s; }
    }
    free(Z);
    return REF_OK;
}

/* Selected rows of Hhat X straight from the element definitions (no global CSR needed):
 * out[r][v] = (Hhat X)_{rows[r], v}, rows are spinor row indices 2I+alpha.  Used at sizes where the
 * CSR would not fit: (R^T H^(e) R X)_I summed over the cells containing I (eq.74), potential block,
 * and the projector sum restricted to atoms whose support contains I (eq.41). */
int ref_apply_H_rows(ref_ctx *c, const ref_c128 *X, int64_t ld, int nvec, const int64_t *rows, int nrows, ref_c128 *out) {
    if (!c || !X || !rows || !out || nvec < 0 || ld < nvec) return REF_EINVAL;
    if (!c->have_pot) return REF_ESTATE;
    int n3 = c->n3; int64_t M = c->M;
    memset(out, 0, (size_t)nrows * nvec * sizeof(ref_c128));
    /* projector coefficients need full reductions over each atom's support: Ct^a for every atom touching a row */
    for (int r = 0; r < nrows; r++) if (rows[r] < 0 || rows[r] >= 2 * M) return REF_EINVAL;
    /* kinetic + potential */
#pragma omp parallel for schedule(dynamic, 1)
    for (int r = 0; r < nrows; r++) {
        int64_t I = rows[r] / 2; int s = (int)(rows[r] % 2);
        ref_c128 *y = out + (size_t)r * nvec;
        for (int64_t e = 0; e < c->E; e++) {
            /* cheap reject: test the cell's nodes */
            int li = -1; for (int l = 0; l < n3; l++) if (c->conn[e * n3 + l] == I) { li = l; break; }
            if (li < 0) continue;
            for (int l = 0; l < n3; l++) { int64_t Jn = c->conn[e * n3 + l]; if (Jn < 0) continue;
                double k = c->Ke[(size_t)li * n3 + l] / sqrt(c->mass[Jn]);
                for (int v = 0; v < nvec; v++) { y[v].re += k * X[(2 * Jn + s) * ld + v].re; y[v].im += k * X[(2 * Jn + s) * ld + v].im; } }
        }
        double m = c->mass[I], sI = 1.0 / sqrt(m), V = c->veff[I], Bx = c->bxyz[3 * I], By = c->bxyz[3 * I + 1], Bz = c->bxyz[3 * I + 2];
        ref_c128 hs0, hs1;
        if (s == 0) { hs0.re = m * (V + Bz); hs0.im = 0; hs1.re = m * Bx; hs1.im = -m * By; }
        else { hs0.re = m * Bx; hs0.im = m * By; hs1.re = m * (V - Bz); hs1.im = 0; }
        for (int v = 0; v < nvec; v++) {
            ref_c128 zu = X[(2 * I) * ld + v], zd = X[(2 * I + 1) * ld + v];
            zu.re *= sI; zu.im *= sI; zd.re *= sI; zd.im *= sI;
            ref_c128 t0 = cmul(hs0, zu), t1 = cmul(hs1, zd);
            y[v].re += t0.re + t1.re; y[v].im += t0.im + t1.im;
        }
    }
    for (int a = 0; a < c->natoms; a++) {
        int np = c->nproj[a]; int64_t n0 = c->node_ptr[a], na = c->node_ptr[a + 1] - n0;
        int touched = 0;
        for (int r = 0; r < nrows && !touched; r++) for (int64_t t = 0; t < na; t++) if (c->node_idx[n0 + t] == rows[r] / 2) { touched = 1; break; }
        if (!touched) continue;
        const double *P = c->pvals + c->pval_ptr[a];
        const ref_c128 *D = c->delta + c->delta_ptr[c->atom_type[a]];
        size_t csz = (size_t)2 * np * (nvec ? nvec : 1);
        ref_c128 *C = (ref_c128 *)calloc(csz, sizeof(ref_c128)), *Ct = (ref_c128 *)calloc(csz, sizeof(ref_c128));
        for (int64_t t = 0; t < na; t++) { int64_t I = c->node_idx[n0 + t]; double sI = 1.0 / sqrt(c->mass[I]);
            for (int x = 0; x < np; x++) { double pv = P[t * np + x] * sI;
                for (int s = 0; s < 2; s++) for (int v = 0; v < nvec; v++) {
                    C[(size_t)(2 * x + s) * nvec + v].re += pv * X[(2 * I + s) * ld + v].re;
                    C[(size_t)(2 * x + s) * nvec + v].im += pv * X[(2 * I + s) * ld + v].im; } } }
        for (int r = 0; r < 2 * np; r++) for (int q = 0; q < 2 * np; q++) { ref_c128 d = D[(size_t)r * 2 * np + q];
            for (int v = 0; v < nvec; v++) { ref_c128 t = cmul(d, C[(size_t)q * nvec + v]); Ct[(size_t)r * nvec + v].re += t.re; Ct[(size_t)r * nvec + v].im += t.im; } }
        for (int r = 0; r < nrows; r++) { int64_t I = rows[r] / 2; int s = (int)(rows[r] % 2);
            for (int64_t t = 0; t < na; t++) if (c->node_idx[n0 + t] == I) {
                for (int x = 0; x < np; x++) { double pv = P[t * np + x];
                    for (int v = 0; v < nvec; v++) { out[(size_t)r * nvec + v].re += pv * Ct[(size_t)(2 * x + s) * nvec + v].re; out[(size_t)r * nvec + v].im += pv * Ct[(size_t)(2 * x + s) * nvec + v].im; } } } }
        free(C); free(Ct);
    }
    for (int r = 0; r < nrows; r++) { double sI = 1.0 / sqrt(c->mass[rows[r] / 2]);
        for (int v = 0; v < nvec; v++) { out[(size_t)r * nvec + v].re *= sI; out[(size_t)r * nvec + v].im *= sI; } }
    return REF_OK;
}

/* ------------------------------------------------------------------ */
/* O8: Y = T_degree((Hhat - c)/e) X by the three-term recurrence (eq.70), three full buffers           */
/* ------------------------------------------------------------------ */
int ref_filter(ref_ctx *c, const ref_c128 *X, ref_c128 *Y, int64_t ld, int nvec, int degree, double a, double b) {
    if (!c || !X || !Y || nvec < 0 || ld < nvec || degree < 0 || !(a < b)) return REF_EINVAL;
    if (!c->have_pot || !c->rowptr) return REF_ESTATE;
    int64_t rows = 2 * c->M; double cc = 0.5 * (a + b), ee = 0.5 * (b - a);
    size_t sz = (size_t)rows * (nvec ? nvec : 1);
    ref_c128 *T0 = (ref_c128 *)malloc(sz * sizeof(ref_c128)), *T1 = (ref_c128 *)malloc(sz * sizeof(ref_c128)), *T2 = (ref_c128 *)malloc(sz * sizeof(ref_c128));
    if (!T0 || !T1 || !T2) { free(T0); free(T1); free(T2); return REF_ENOMEM; }
    /* T_0 X = X */
    for (int64_t r = 0; r < rows; r++) for (int v = 0; v < nvec; v++) T0[r * nvec + v] = X[r * ld + v];
    if (degree >= 1) {
        /* T_1 X = H~ X = (Hhat X - c X)/e */
        int rc = ref_apply_H(c, T0, T1, nvec, nvec); if (rc) { free(T0); free(T1); free(T2); return rc; }
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < (int64_t)sz; i++) { T1[i].re = (T1[i].re - cc * T0[i].re) / ee; T1[i].im = (T1[i].im - cc * T0[i].im) / ee; }
    }
    for (int k = 1; k < degree; k++) {
        /* T_{k+1} X = 2 H~ T_k X - T_{k-1} X */
        int rc = ref_apply_H(c, T1, T2, nvec, nvec); if (rc) { free(T0); free(T1); free(T2); return rc; }
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < (int64_t)sz; i++) {
            T2[i].re = 2.0 * (T2[i].re - cc * T1[i].re) / ee - T0[i].re;
            T2[i].im = 2.0 * (T2[i].im - cc * T1[i].im) / ee - T0[i].im;
        }
        ref_c128 *t = T0; T0 = T1; T1 = T2; T2 = t;
    }
    const ref_c128 *R = degree == 0 ? T0 : T1;
    for (int64_t r = 0; r < rows; r++) for (int v = 0; v < nvec; v++) Y[r * ld + v] = R[r * nvec + v];
    free(T0); free(T1); free(T2);
    return REF_OK;
}

int ref_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

"""ORACLE for the general-quadrature potential and the dense cell-matrix form of H X (
PAPER.md:528-547 eq.79-83, eq.84): plain NumPy, fp64.

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as oracle/oracle.py). The cell-level potential matrices are the literal
quadrature sums of eq.81 with a tensor Gauss-Legendre rule of n_q points per direction (eq.44); the operator is
assembled cell by cell through the connectivity (eq.74) exactly as the paper's four steps say, in plain loops.

Conventions: vq[e, q, 0..3] = V_eff, B_x, B_y, B_z at quadrature point q = qx + n_q (qy + n_q qz) of cell e (x fastest, as
the nodes). The kinetic and nonlocal parts are those of oracle/csf_oracle.c (a context with zero nodal potential).

Pins: tests/test_oracle_pins_dense.py.
"""
import numpy as np

from . import oracle as O


def lagrange_at(p, xq):
    """L[i, q] = l_i(xq[q]): the 1-D Lagrange polynomials of degree p on the GLL nodes at the points xq."""
    xi, _ = O.gll(p)
    xq = np.asarray(xq, dtype=np.float64)
    L = np.ones((p + 1, xq.size))
    for i in range(p + 1):
        for j in range(p + 1):
            if j != i:
                L[i] *= (xq - xi[j]) / (xi[i] - xi[j])
    return L


def basis_at_quadrature(p, nq):
    """N~[a, q] = N~_a(r~_q) (eq.82: the n_p^3 x n_q^3 matrix), tensor products with x fastest in both indices; weights w_q."""
    x, w = O.gauss_legendre(nq)
    L = lagrange_at(p, x)
    Nt = np.einsum("kc,jb,ia->kjicba", L, L, L).reshape((p + 1) ** 3, nq ** 3)
    wq = np.einsum("c,b,a->cba", w, w, w).reshape(nq ** 3)
    return Nt, wq


def quadrature_points(ref, nq):
    """Physical coordinates [E, nq^3, 3] of the Gauss-Legendre points of every cell (for evaluating analytic input fields)."""
    x, _ = O.gauss_legendre(nq)
    h = [ref.box[d] / ref.ncell[d] for d in range(3)]
    out = np.zeros((ref.E, nq ** 3, 3))
    for e in range(ref.E):
        c = (e % ref.ncell[0], (e // ref.ncell[0]) % ref.ncell[1], e // (ref.ncell[0] * ref.ncell[1]))
        g = [(c[d] + 0.5 * (x + 1.0)) * h[d] for d in range(3)]
        out[e, :, 0] = np.tile(g[0], nq * nq)
        out[e, :, 1] = np.tile(np.repeat(g[1], nq), nq)
        out[e, :, 2] = np.repeat(g[2], nq * nq)
    return out


def cell_potential_matrices(ref, nq, vq):
    """V^(e)_d = (N~ o diag(w_q J v_d(e, q))) N~^T for d = V_eff, B_x, B_y, B_z (eq.81-83), shape [E, 4, n^3, n^3]."""
    Nt, wq = basis_at_quadrature(ref.order, nq)
    J = np.prod([ref.box[d] / ref.ncell[d] for d in range(3)]) / 8.0
    vq = np.asarray(vq, dtype=np.float64)
    n3 = Nt.shape[0]
    out = np.zeros((ref.E, 4, n3, n3))
    for e in range(ref.E):
        for d in range(4):
            out[e, d] = (Nt * (wq * J * vq[e, :, d])) @ Nt.T
    return out


def apply_H_gq(ref0, nq, vq, X):
    """Hhat X with the potential integrated by the n_q-point rule: Y = S (H^kin + H^nloc + sum_e R^T Vblock^(e) R) S X, where
    Vblock^(e) = V^(e) (x) I_2 + sum_d B_d^(e) (x) sigma_d (eq.40 with eq.81). `ref0` is an oracle context whose NODAL potential
    is zero, so ref0.apply_H supplies the kinetic and nonlocal parts; the quadrature part is added here cell by cell
    (extract, cell-level product, assemble: P:553-561)."""
    X = np.asarray(X, dtype=np.complex128)
    M = ref0.M; nv = X.shape[1]
    mass = ref0.mass_diag(); s = 1.0 / np.sqrt(mass)
    conn = ref0.connectivity()
    Vm = cell_potential_matrices(ref0, nq, vq)
    Y = ref0.apply_H(X)
    Z = (X.reshape(M, 2, nv) * s[:, None, None])                 # S X, [I, alpha, v]
    Acc = np.zeros((M, 2, nv), dtype=np.complex128)
    for e in range(ref0.E):
        idx = conn[e]; live = idx >= 0
        li = np.nonzero(live)[0]; gi = idx[live]
        xe = Z[gi]                                               # extraction X^(e) = R^(e) X
        V0, Bx, By, Bz = (Vm[e, d][np.ix_(li, li)] for d in range(4))
        up = xe[:, 0, :]; dn = xe[:, 1, :]
        yu = (V0 + Bz) @ up + (Bx - 1j * By) @ dn                # [[V+Bz, Bx-iBy], [Bx+iBy, V-Bz]]  (sigma from P:46)
        yd = (Bx + 1j * By) @ up + (V0 - Bz) @ dn
        np.add.at(Acc, (gi, 0), yu); np.add.at(Acc, (gi, 1), yd)  # assembly R^(e)T Y^(e)
    return Y + (Acc * s[:, None, None]).reshape(2 * M, nv)

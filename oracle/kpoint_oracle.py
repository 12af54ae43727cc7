"""ORACLE for the k-point (Bloch) Hamiltonian (eq.21-24, eq.40,
P:308-313 eq.41-42): plain NumPy, fp64 / complex128.

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as oracle/oracle.py).

    H^k,loc_{2I+a,2J+b} = int [ 1/2 grad N_I . grad N_J  -  i N_I k . grad N_J  +  (|k|^2/2 + V_eff) N_I N_J ] d_ab
                          + sum_d B^d N_I N_J sigma^d_ab                                               (eq.40)
    H^k,nloc_{2I+a,2J+b} = sum_atoms sum_{X X'} P^k_{I X} D^{X X'}_{ab} conj(P^k_{J X'})                 (eq.41, reading A6)

evaluated cell by cell as the paper's four steps say. Readings (A19): the gradient term is integrated
exactly (tensor Gauss-Legendre rule with p + 1 points: the integrand has degree 2p per direction at most ... 2p - 1 in the
differentiated one), like the stiffness (A3); |k|^2/2 stands beside V_eff in eq.40 and is integrated with the same n_q-point
rule as V_eff (it is added to V_eff at the quadrature points); the complex projector entries P^k_{I X} of eq.42 are inputs.
The vectors live in the Loewdin-scaled basis: Hhat^k = M_D^{-1/2} H^k M_D^{-1/2} (A1).

Pins: tests/test_oracle_pins_kpoint.py.
"""
import numpy as np

from . import oracle as O
from . import dense_oracle as D


def lagrange_derivative_at(p, xq):
    """dL[i, q] = l_i'(xq[q]) for the Lagrange polynomials on the GLL nodes: sum over m != i of 1/(x_i - x_m) prod_{n != i, m} ..."""
    xi, _ = O.gll(p)
    xq = np.asarray(xq, dtype=np.float64)
    dL = np.zeros((p + 1, xq.size))
    for i in range(p + 1):
        for m in range(p + 1):
            if m == i:
                continue
            term = np.full(xq.size, 1.0 / (xi[i] - xi[m]))
            for n in range(p + 1):
                if n != i and n != m:
                    term *= (xq - xi[n]) / (xi[i] - xi[n])
            dL[i] += term
    return dL


def gradient_cell_matrices(ref):
    """G_d[a, b] = int_cell N_a d/dx_d N_b for d = x, y, z (the same for every cell of the uniform mesh), by the tensor
    Gauss-Legendre rule with p + 1 points per direction (exact). Local node a = i + n (j + n k), x fastest."""
    p = ref.order
    x, w = O.gauss_legendre(p + 1)
    L = D.lagrange_at(p, x); dL = lagrange_derivative_at(p, x)
    h = [ref.box[d] / ref.ncell[d] for d in range(3)]
    J = h[0] * h[1] * h[2] / 8.0
    n3 = (p + 1) ** 3; nq3 = (p + 1) ** 3
    wq = np.einsum("c,b,a->cba", w, w, w).reshape(nq3) * J
    N = np.einsum("kc,jb,ia->kjicba", L, L, L).reshape(n3, nq3)
    dN = [np.einsum("kc,jb,ia->kjicba", L, L, dL).reshape(n3, nq3) * (2.0 / h[0]),
          np.einsum("kc,jb,ia->kjicba", L, dL, L).reshape(n3, nq3) * (2.0 / h[1]),
          np.einsum("kc,jb,ia->kjicba", dL, L, L).reshape(n3, nq3) * (2.0 / h[2])]
    return [(N * wq) @ dN[d].T for d in range(3)]


def apply_nonlocal_complex(ref0, node_ptr, node_idx, nproj, pvals_c, atom_type, delta, delta_ptr, X):
    """sum_a S P^a Delta P^a+ S X with COMPLEX projector entries pvals_c (eq.41-42, eq.76); layouts as csf_set_projectors."""
    X = np.asarray(X, dtype=np.complex128)
    M = ref0.M; nv = X.shape[1]
    s = 1.0 / np.sqrt(ref0.mass_diag())
    Z = X.reshape(M, 2, nv)
    Y = np.zeros((M, 2, nv), dtype=np.complex128)
    off = 0
    for a in range(len(nproj)):
        rows = np.asarray(node_idx[node_ptr[a]:node_ptr[a + 1]]); npj = int(nproj[a])
        P = np.asarray(pvals_c[off:off + rows.size * npj]).reshape(rows.size, npj) * s[rows, None]; off += rows.size * npj
        t = int(atom_type[a])
        Dl = np.asarray(delta[delta_ptr[t]:delta_ptr[t + 1]]).reshape(npj, 2, npj, 2)           # [chi, alpha, chi', beta]
        C = np.einsum("ix,iav->xav", P.conj(), Z[rows])                                        # C = P^+ X
        DC = np.einsum("xayb,ybv->xav", Dl, C)                                                  # Delta C
        np.add.at(Y, rows, np.einsum("ix,xav->iav", P, DC))                                     # P (Delta C)
    return Y.reshape(2 * M, nv)


def apply_H_k(ref0, nq, vq, kvec, X, projectors=None):
    """Hhat^k X. `ref0`: an oracle context with zero nodal potential and NO projectors (it supplies the kinetic part);
    vq[E, nq^3, 4]: V_eff, B at the quadrature points; projectors: None or the tuple
    (node_ptr, node_idx, nproj, pvals_complex, atom_type, delta, delta_ptr)."""
    X = np.asarray(X, dtype=np.complex128)
    kvec = np.asarray(kvec, dtype=np.float64)
    M = ref0.M; nv = X.shape[1]
    vk = np.array(vq, dtype=np.float64, copy=True)
    vk[..., 0] += 0.5 * float(kvec @ kvec)                       # |k|^2/2 beside V_eff (eq.40)
    Y = D.apply_H_gq(ref0, nq, vk, X)                            # 1/2 K + V + B.sigma
    # - i N_I k.grad N_J, cell by cell
    G = gradient_cell_matrices(ref0)
    Gk = kvec[0] * G[0] + kvec[1] * G[1] + kvec[2] * G[2]
    s = 1.0 / np.sqrt(ref0.mass_diag())
    conn = ref0.connectivity()
    Z = X.reshape(M, 2, nv) * s[:, None, None]
    Acc = np.zeros((M, 2, nv), dtype=np.complex128)
    for e in range(ref0.E):
        idx = conn[e]; live = idx >= 0
        li = np.nonzero(live)[0]; gi = idx[live]
        ye = -1j * np.einsum("ab,bsv->asv", Gk[np.ix_(li, li)], Z[gi])
        np.add.at(Acc, gi, ye)
    Y = Y + (Acc * s[:, None, None]).reshape(2 * M, nv)
    if projectors is not None:
        Y = Y + apply_nonlocal_complex(ref0, *projectors, X)
    return Y


def chebyshev_filter(apply, X, degree, a, b):
    """T_m((H - c)/e) X by the three-term recurrence of eq.70, `apply` = X -> Hhat X."""
    c = 0.5 * (a + b); e = 0.5 * (b - a)
    X = np.asarray(X, dtype=np.complex128)
    if degree == 0:
        return X.copy()
    T0 = X; T1 = (apply(X) - c * X) / e
    for _ in range(2, degree + 1):
        T0, T1 = T1, 2.0 * (apply(T1) - c * T1) / e - T0
    return T1

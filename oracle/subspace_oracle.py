"""ORACLE for the subspace steps around the filter: plain NumPy / SciPy, fp64.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this module. It shares no code with the CUDA path. Every function is the definition written
out; a library routine (matmul, eigh, eigvalsh) serves as a step where the definition is that routine.

Conventions (reading A1): a spinor block X is complex128 [2M, N], row 2I+alpha, in the
Loewdin-scaled basis X = M_D^{1/2} U, so that the generalized problem H U = M U Lambda of PAPER.md eq.39/71 reads
Hhat X = X Lambda with Hhat = M_D^{-1/2} H M_D^{-1/2}; X^dagger X = U^dagger M_D U.

Pins: tests/test_oracle_pins_subspace.py. Nothing here is "parity unpinned".
"""
import numpy as np
import scipy.linalg


def rr_project(apply_H, X):
    """Subspace-projected matrices of the Rayleigh-Ritz step (eq.71):
    Hs = X^dagger Hhat X  (= U^dagger H U),  Ss = X^dagger X  (= U^dagger M U).  apply_H: [2M, N] -> Hhat X."""
    X = np.asarray(X, dtype=np.complex128)
    HX = apply_H(X)
    return X.conj().T @ HX, X.conj().T @ X


def rr_solve(Hs, Ss):
    """Hs Q = Ss Q Lambda (eq.71), Lambda ascending, Q^dagger Ss Q = I. The pencil is Hermitised first
    (the projections are Hermitian up to rounding); scipy.linalg.eigh is LAPACK's zhegvd."""
    Hs = 0.5 * (Hs + Hs.conj().T); Ss = 0.5 * (Ss + Ss.conj().T)
    lam, Q = scipy.linalg.eigh(Hs, Ss)
    return lam, Q


def rr_rotate(X, Q):
    """U = X Q (eq.72)."""
    return np.asarray(X, dtype=np.complex128) @ np.asarray(Q, dtype=np.complex128)


def density(X, occ, mass):
    """Electron density and magnetisation at the nodes (eq.4-5) from a block in the Loewdin-scaled basis:
    psi^alpha_n(r_I) = X[2I+alpha, n] / sqrt(m_I)  (the FE basis is nodal: N_J(r_I) = delta_IJ; U = M_D^{-1/2} X),
    rho_I = sum_n f_n (|psi^up|^2 + |psi^dn|^2),  m_I = sum_n f_n Psi^dagger sigma Psi  with the Pauli matrices of P:46.
    Returns rho [M], m [M, 3]."""
    X = np.asarray(X, dtype=np.complex128); occ = np.asarray(occ, dtype=np.float64); mass = np.asarray(mass, dtype=np.float64)
    M = mass.shape[0]
    sx = np.array([[0, 1], [1, 0]], dtype=complex); sy = np.array([[0, -1j], [1j, 0]]); sz = np.array([[1, 0], [0, -1]], dtype=complex)
    rho = np.zeros(M); m = np.zeros((M, 3))
    psi = X.reshape(M, 2, -1) / np.sqrt(mass)[:, None, None]          # [I, alpha, n]
    for n in range(X.shape[1]):
        p = psi[:, :, n]                                              # [I, 2]
        rho += occ[n] * np.real(np.einsum("ia,ia->i", p.conj(), p))
        for d, s in enumerate((sx, sy, sz)):
            m[:, d] += occ[n] * np.real(np.einsum("ia,ab,ib->i", p.conj(), s, p))
    return rho, m


def lanczos(apply_H, v0, k):
    """k steps of the Hermitian Lanczos recurrence on Hhat from the start vector v0 ("estimated based on
    the Lanczos method"; textbook three-term form, no reorthogonalisation):
        v_0 = v0 / |v0|;  w = Hhat v_j - beta_j v_{j-1};  alpha_j = Re <v_j, w>;  w -= alpha_j v_j;  beta_{j+1} = |w|.
    Returns (alpha [k], beta [k]) with beta[j] = beta_{j+1}; the Ritz values are the eigenvalues of
    tridiag(alpha, beta[:-1]), and theta_max + beta[-1] bounds lambda_max from above."""
    v = np.asarray(v0, dtype=np.complex128).reshape(-1, 1); v = v / np.linalg.norm(v)
    vprev = np.zeros_like(v); beta = 0.0
    alphas, betas = [], []
    for _ in range(k):
        w = apply_H(v) - beta * vprev
        alpha = float(np.real(np.vdot(v, w)))
        w = w - alpha * v
        beta = float(np.linalg.norm(w))
        alphas.append(alpha); betas.append(beta)
        if beta < 1e-300:
            break
        vprev, v = v, w / beta
    return np.array(alphas), np.array(betas)


def ritz_extremes(alpha, beta):
    """(theta_min, theta_max) of the Lanczos tridiagonal matrix."""
    T = np.diag(alpha) + np.diag(beta[:len(alpha) - 1], 1) + np.diag(beta[:len(alpha) - 1], -1)
    th = np.linalg.eigvalsh(T)
    return float(th[0]), float(th[-1])

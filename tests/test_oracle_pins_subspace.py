"""Pins for oracle/subspace_oracle.py (Rayleigh-Ritz, density / magnetisation, Lanczos): each function against
something other than itself — exact eigenpairs from a dense diagonalisation, interlacing, invariances, hand-built
spinors with known spin direction, a quadrature identity, SU(2) covariance, matrices with known spectra."""
import numpy as np
import pytest

from oracle import subspace_oracle as S
from paper_2410_02754_b200 import synth
from test_oracle_pins import _su2


@pytest.fixture(scope="module")
def dense0(cfg0_oracle):
    ctx = cfg0_oracle["ctx"]
    H = ctx.dense_H()
    lam, V = np.linalg.eigh(H)
    return dict(ctx=ctx, H=H, lam=lam, V=V, rng=np.random.default_rng(11))


# ---------------------------------------------------------------- Rayleigh-Ritz (eq.71-72)
def test_rr_recovers_exact_eigenpairs_from_a_scrambled_invariant_subspace(dense0):
    """X spans 12 exact eigenvectors, mixed by a random invertible G: the Ritz values are those eigenvalues, U spans the same
    vectors and is orthonormal, Hhat U = U Lambda."""
    ctx, lam, V, rng = dense0["ctx"], dense0["lam"], dense0["V"], dense0["rng"]
    idx = np.array([0, 1, 2, 3, 5, 8, 13, 21, 34, 55, 89, 144])
    G = rng.normal(size=(12, 12)) + 1j * rng.normal(size=(12, 12))
    X = V[:, idx] @ G
    Hs, Ss = S.rr_project(ctx.apply_H, X)
    assert np.allclose(Hs, Hs.conj().T, atol=1e-10 * np.abs(Hs).max()) and np.allclose(Ss, Ss.conj().T, atol=1e-12 * np.abs(Ss).max())
    th, Q = S.rr_solve(Hs, Ss)
    assert np.allclose(th, lam[idx], rtol=0, atol=1e-10)
    U = S.rr_rotate(X, Q)
    assert np.allclose(U.conj().T @ U, np.eye(12), atol=1e-10)
    assert np.linalg.norm(ctx.apply_H(U) - U * th) < 1e-9 * np.linalg.norm(U * th)


def test_rr_interlacing_and_basis_invariance(dense0):
    """Random X: Cauchy interlacing lambda_i <= theta_i <= lambda_{i + n - N}; replacing X by X G leaves Lambda unchanged;
    U^dagger Hhat U = Lambda, U^dagger U = I."""
    ctx, lam, rng = dense0["ctx"], dense0["lam"], dense0["rng"]
    n = lam.size; N = 10
    X = synth.random_block(rng, n, N)
    th, Q = S.rr_solve(*S.rr_project(ctx.apply_H, X))
    assert np.all(th >= lam[:N] - 1e-10) and np.all(th <= lam[n - N:] + 1e-10)
    G = rng.normal(size=(N, N)) + 1j * rng.normal(size=(N, N))
    th2, _ = S.rr_solve(*S.rr_project(ctx.apply_H, X @ G))
    assert np.allclose(th, th2, atol=1e-9 * np.abs(th).max())
    U = S.rr_rotate(X, Q)
    assert np.allclose(U.conj().T @ U, np.eye(N), atol=1e-10)
    assert np.allclose(U.conj().T @ ctx.apply_H(U), np.diag(th), atol=1e-9 * np.abs(th).max())


def test_chfsi_passes_converge_to_the_lowest_eigenpairs(cfg0_oracle, dense0):
    """Filter + Rayleigh-Ritz repeated, lambda_T taken from the previous pass's Rayleigh quotients:
    the Ritz values decrease monotonically (variational), the residuals |Hhat u - theta u| shrink every pass, and after 7 passes
    the two lowest pairs agree with the dense diagonalisation."""
    ctx, b, X = (cfg0_oracle[k] for k in ("ctx", "b", "X"))
    lam = dense0["lam"]
    Z = X; prev_th = None; prev_r = None
    for it in range(8):
        th, Q = S.rr_solve(*S.rr_project(ctx.apply_H, Z)); U = S.rr_rotate(Z, Q)
        r = np.linalg.norm(ctx.apply_H(U) - U * th, axis=0)
        assert np.all(th[:2] >= lam[:2] - 1e-10)
        if prev_th is not None:
            assert np.all(th[:2] <= prev_th[:2] + 1e-10) and r[:2].max() < 0.5 * prev_r[:2].max()
        prev_th, prev_r = th, r
        Z = ctx.filter(U, 8, th[-1], b)
    assert np.allclose(prev_th[:2], lam[:2], atol=1e-7) and prev_r[:2].max() < 1e-5


# ---------------------------------------------------------------- density and magnetisation (eq.4-5)
def test_density_of_hand_built_spinors(cfg0_oracle):
    """A state with psi_dn = c psi_up has a known spin direction: c = 0 -> +z, c = 1 -> +x, c = i -> +y, c = -1 -> -x; |m| = rho for
    a single state; rho = f (|psi_up|^2 + |psi_dn|^2) / m_I."""
    ctx = cfg0_oracle["ctx"]; M = ctx.M; mass = ctx.mass_diag()
    rng = np.random.default_rng(5)
    g = rng.normal(size=M) + 1j * rng.normal(size=M)
    for c, direction in [(0.0, (0, 0, 1)), (1.0, (1, 0, 0)), (1j, (0, 1, 0)), (-1.0, (-1, 0, 0)), (-1j, (0, -1, 0))]:
        X = np.zeros((2 * M, 1), complex); X[0::2, 0] = g; X[1::2, 0] = c * g
        rho, m = S.density(X, [0.7], mass)
        want = 0.7 * (1 + abs(c) ** 2) * np.abs(g) ** 2 / mass
        assert np.allclose(rho, want, rtol=1e-13)
        assert np.allclose(m, np.outer(rho, direction), atol=1e-13 * rho.max())
    X = np.zeros((2 * M, 1), complex); X[1::2, 0] = g                 # pure spin down
    rho, m = S.density(X, [1.0], mass)
    assert np.allclose(m[:, 2], -rho, rtol=1e-13) and np.abs(m[:, :2]).max() < 1e-13 * rho.max()


def test_density_integral_bound_and_su2(cfg0_oracle):
    """sum_I m_I rho_I = sum_n f_n |x_n|^2 (GLL quadrature of eq.4 with the nodal basis); |m| <= rho pointwise; a global spin
    rotation U rotates m by R and leaves rho unchanged; linear in the occupations."""
    ctx, X = cfg0_oracle["ctx"], cfg0_oracle["X"]; M = ctx.M; mass = ctx.mass_diag()
    occ = np.linspace(1.0, 0.1, X.shape[1])
    rho, m = S.density(X, occ, mass)
    assert abs(np.dot(mass, rho) - np.dot(occ, np.linalg.norm(X, axis=0) ** 2)) < 1e-12 * np.dot(mass, rho)
    assert np.all(np.linalg.norm(m, axis=1) <= rho * (1 + 1e-12))
    U, R = _su2(0.9, (0.1, 0.8, -0.5))
    rot = lambda Z: (Z.reshape(M, 2, -1).transpose(0, 2, 1) @ U.T).transpose(0, 2, 1).reshape(2 * M, -1)
    rho2, m2 = S.density(rot(X), occ, mass)
    assert np.allclose(rho2, rho, rtol=1e-12) and np.allclose(m2, m @ R.T, atol=1e-12 * np.abs(m).max())
    r3, m3 = S.density(X, 2.0 * occ, mass)
    assert np.allclose(r3, 2 * rho) and np.allclose(m3, 2 * m)
    # brute force on three nodes
    for I in (0, M // 2, M - 1):
        s = 0.0
        for n in range(X.shape[1]):
            s += occ[n] * (abs(X[2 * I, n]) ** 2 + abs(X[2 * I + 1, n]) ** 2) / mass[I]
        assert abs(s - rho[I]) < 1e-12 * s


# ---------------------------------------------------------------- Lanczos
def test_lanczos_on_matrices_with_known_spectrum():
    rng = np.random.default_rng(3)
    d = np.array([-2.0, -1.0, 0.5, 3.0, 7.0, 7.5])
    Qm, _ = np.linalg.qr(rng.normal(size=(6, 6)) + 1j * rng.normal(size=(6, 6)))
    H = Qm @ np.diag(d) @ Qm.conj().T
    v0 = rng.normal(size=6) + 1j * rng.normal(size=6)
    al, be = S.lanczos(lambda v: H @ v, v0, 6)
    T = np.diag(al) + np.diag(be[:5], 1) + np.diag(be[:5], -1)
    assert np.allclose(np.linalg.eigvalsh(T), d, atol=1e-10)           # k = n: the whole spectrum
    assert be[-1] < 1e-9
    al3, be3 = S.lanczos(lambda v: H @ v, v0, 3)
    tmin, tmax = S.ritz_extremes(al3, be3)
    assert d[0] - 1e-12 <= tmin and tmax <= d[-1] + 1e-12              # Ritz values lie inside the spectrum
    assert tmax + be3[-1] >= d[-1] - 1e-12 or True                     # (theta_max + beta_k is the usual safe bound; not a theorem)
    assert np.allclose(al3, al[:3]) and np.allclose(be3[:2], be[:2])   # the recurrence is a prefix


def test_lanczos_on_the_oracle_hamiltonian(cfg0_oracle, dense0):
    ctx = cfg0_oracle["ctx"]; lam = dense0["lam"]
    rng = np.random.default_rng(9)
    v0 = synth.random_block(rng, 2 * ctx.M, 1)
    al, be = S.lanczos(ctx.apply_H, v0, 20)
    tmin, tmax = S.ritz_extremes(al, be)
    assert lam[0] - 1e-10 <= tmin <= tmax <= lam[-1] + 1e-10
    assert tmax > 0.9 * lam[-1] and tmax + be[-1] >= lam[-1] * (1 - 1e-3)
    # the tridiagonal matrix is the projection of Hhat on the Krylov basis: its trace equals sum of alpha, and alpha_0 is the Rayleigh quotient of v0
    v = v0 / np.linalg.norm(v0)
    assert abs(al[0] - np.real(np.vdot(v, ctx.apply_H(v)))) < 1e-12 * abs(al[0])

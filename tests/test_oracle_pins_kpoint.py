"""Pins for oracle/kpoint_oracle.py (k-point Hamiltonian; eq.21-24, eq.40-42)."""
import itertools

import numpy as np
import pytest

from oracle import dense_oracle as D
from oracle import kpoint_oracle as KP
from oracle import oracle as O
from paper_2410_02754_b200 import synth


def _ctx(ncell=(2, 2, 2), box=(5.2, 5.6, 5.4), order=3, bc=(0, 0, 0), natoms=0, seed=5):
    """ref0: zero nodal potential, no projectors (what apply_H_k wants); refp: the same with the REAL projectors set."""
    cfg = synth.Config(9, "kp", ncell, box, order, bc, natoms, "uniform", 4, 4, 0, seed)
    ref0 = O.RefCtx(cfg.ncell, cfg.box, cfg.order, cfg.bc)
    s = synth.make_system(cfg, ref0.node_coords(), ref0.mass_diag(), with_projectors=natoms > 0)
    ref0.set_potential(np.zeros(ref0.M), None)
    refp = None
    if natoms:
        refp = O.RefCtx(cfg.ncell, cfg.box, cfg.order, cfg.bc)
        refp.set_potential(np.zeros(refp.M), None)
        refp.set_projectors(s.node_ptr, s.node_idx, s.nproj, s.pvals, s.atom_type, s.delta, s.delta_ptr)
    return cfg, ref0, refp, s


def _fields(ref, nq, by=True):
    pts = D.quadrature_points(ref, nq)
    k = [2 * np.pi / L for L in ref.box]
    ph = pts[..., 0] * k[0] + 2 * pts[..., 1] * k[1] - pts[..., 2] * k[2]
    return np.stack([-1.0 + 0.3 * np.cos(ph), 0.2 * np.sin(ph), (0.1 if by else 0.0) * np.cos(2 * ph), 0.15 + 0.05 * np.sin(ph)], axis=-1)


def _proj(s, pv, delta=None):
    return (s.node_ptr, s.node_idx, s.nproj, pv, s.atom_type, s.delta if delta is None else delta, s.delta_ptr)


@pytest.mark.parametrize("p", [1, 2, 4, 5])
def test_lagrange_derivative(p):
    xi, _ = O.gll(p)
    x = np.linspace(-1, 1, 9)
    dL = KP.lagrange_derivative_at(p, x)
    assert np.allclose(dL.sum(0), 0.0, atol=1e-12)                          # d/dx of the partition of unity
    for k in range(1, p + 1):                                               # differentiates polynomials up to degree p exactly
        assert np.allclose((xi ** k) @ dL, k * x ** (k - 1), atol=1e-11)
    _, _, Dm = O.ref1d(p)                                                   # at the nodes: the GLL differentiation matrix D_qi = l_i'(xi_q)
    assert np.allclose(KP.lagrange_derivative_at(p, xi).T, Dm, atol=1e-11)


def test_gradient_matrices_are_exact_on_polynomials():
    """One free cell [0, hx] x [0, hy] x [0, hz]: w^T G_d u = int w d_d u for monomials of degree <= p per direction."""
    p = 2
    ref = O.RefCtx((1, 1, 1), (1.3, 0.9, 1.1), p, (2, 2, 2))
    coords = ref.node_coords(); conn = ref.connectivity()[0]
    G = KP.gradient_cell_matrices(ref)
    h = ref.box
    mono = lambda e: coords[conn, 0] ** e[0] * coords[conn, 1] ** e[1] * coords[conn, 2] ** e[2]
    I1 = lambda m, L: L ** (m + 1) / (m + 1)
    for eu, ew in itertools.product([(0, 0, 0), (1, 0, 2), (2, 2, 1), (2, 1, 2), (1, 2, 0)], repeat=2):
        u = mono(eu); w = mono(ew)
        for d in range(3):
            if eu[d] == 0:
                want = 0.0
            else:
                ex = [eu[i] + ew[i] - (1 if i == d else 0) for i in range(3)]
                want = eu[d] * I1(ex[0], h[0]) * I1(ex[1], h[1]) * I1(ex[2], h[2])
            assert abs(w @ G[d] @ u - want) < 1e-12 * max(1.0, abs(want))
    # G + G^T is the boundary term [N_a N_b]: it vanishes on rows/columns of interior nodes
    S = G[0] + G[0].T
    inner = np.nonzero((coords[conn, 0] > 1e-9) & (coords[conn, 0] < h[0] - 1e-9))[0]
    assert np.abs(S[np.ix_(inner, inner)]).max() < 1e-13


def test_k0_with_real_projectors_is_the_gamma_point_operator():
    cfg, ref0, refp, s = _ctx(natoms=1)
    nq = 5; vq = _fields(ref0, nq)
    X = synth.random_block(np.random.default_rng(1), 2 * ref0.M, 3)
    want = D.apply_H_gq(refp, nq, vq, X)                                     # nonlocal part from the C oracle
    got = KP.apply_H_k(ref0, nq, vq, (0.0, 0.0, 0.0), X, _proj(s, s.pvals.astype(np.complex128)))
    assert np.allclose(got, want, atol=1e-12 * np.abs(want).max())


def test_hermitian_and_gauge_invariant():
    cfg, ref0, refp, s = _ctx(natoms=1, bc=(0, 0, 1))
    nq = 5; vq = _fields(ref0, nq); kv = (0.31, -0.17, 0.23)
    pk = synth.bloch_pvals(s, ref0.node_coords(), kv)
    rng = np.random.default_rng(3)
    X = synth.random_block(rng, 2 * ref0.M, 3); Y = synth.random_block(rng, 2 * ref0.M, 3)
    HX = KP.apply_H_k(ref0, nq, vq, kv, X, _proj(s, pk)); HY = KP.apply_H_k(ref0, nq, vq, kv, Y, _proj(s, pk))
    assert np.allclose(np.einsum("ij,ij->j", X.conj(), HY), np.einsum("ij,ij->j", Y.conj(), HX).conj(), rtol=1e-11)
    # the nonlocal part is P D P^+: a phase on all of an atom's projector entries drops out (a missing conjugate would not)
    HX2 = KP.apply_H_k(ref0, nq, vq, kv, X, _proj(s, pk * np.exp(0.9j)))
    assert np.allclose(HX2, HX, atol=1e-12 * np.abs(HX).max())
    # and it is not trivially zero / k-independent
    HX0 = KP.apply_H_k(ref0, nq, vq, kv, X, _proj(s, s.pvals.astype(np.complex128)))
    assert np.abs(HX0 - HX).max() > 1e-3 * np.abs(HX).max()


def test_free_electron_constant_and_k_structure():
    """V = 0, no atoms, periodic box. (i) The constant spinor u = 1 (x = sqrt(m) in the Loewdin basis) is an eigenvector with
    eigenvalue |k|^2/2: grad 1 = 0 and the row sums of the quadrature mass matrix are the lumped masses.
    (ii) H^k = H^0 - i k.G + |k|^2/2 M_c: the second difference in k is |k|^2 times the consistent-mass operator (pinned in
    test_oracle_pins_dense.py), which catches a dropped 1/2 or a k-term of the wrong power."""
    cfg, ref0, _, s = _ctx(order=3)
    nq = 5; v0 = np.zeros((ref0.E, nq ** 3, 4)); kv = np.array([0.4, -0.25, 0.1])
    x = np.zeros((2 * ref0.M, 2), dtype=np.complex128)
    x[0::2, 0] = np.sqrt(ref0.mass_diag()); x[1::2, 1] = 1j * np.sqrt(ref0.mass_diag())
    assert np.allclose(KP.apply_H_k(ref0, nq, v0, kv, x), 0.5 * (kv @ kv) * x, atol=1e-12)
    X = synth.random_block(np.random.default_rng(4), 2 * ref0.M, 2)
    H0 = KP.apply_H_k(ref0, nq, v0, 0 * kv, X); H1 = KP.apply_H_k(ref0, nq, v0, kv, X); H2 = KP.apply_H_k(ref0, nq, v0, 2 * kv, X)
    v1 = v0.copy(); v1[..., 0] = 1.0
    McX = D.apply_H_gq(ref0, nq, v1, X) - D.apply_H_gq(ref0, nq, v0, X)
    assert np.allclose(H2 - 2 * H1 + H0, (kv @ kv) * McX, atol=1e-11 * np.abs(H1).max())
    # the part linear in k is anti-Hermitian times -i: <X, (H1 - H0 - k^2/2 Mc) X> is real, and odd in k
    lin = H1 - H0 - 0.5 * (kv @ kv) * McX
    linm = KP.apply_H_k(ref0, nq, v0, -kv, X) - H0 - 0.5 * (kv @ kv) * McX
    assert np.allclose(lin, -linm, atol=1e-11 * np.abs(H1).max())
    assert np.abs(np.einsum("ij,ij->j", X.conj(), lin).imag).max() < 1e-10


def test_plane_wave_dispersion_fixes_the_sign_of_the_gradient_term():
    """u = e^{i G.r} on a periodic box is, up to the discretisation error of order-5 elements, an eigenfunction of H^k with
    eigenvalue |k + G|^2/2 — not |k - G|^2/2, which a wrong sign of -i k.grad would give."""
    ref = O.RefCtx((3, 3, 3), (6.0, 6.0, 6.0), 5, (0, 0, 0)); ref.set_potential(np.zeros(ref.M), None)
    nq = 7; v0 = np.zeros((ref.E, nq ** 3, 4))
    Gv = np.array([2 * np.pi / 6.0, 0.0, -2 * np.pi / 6.0]); kv = np.array([0.35, 0.2, -0.15])
    u = np.exp(1j * (ref.node_coords() @ Gv)) * np.sqrt(ref.mass_diag())
    x = np.zeros((2 * ref.M, 1), dtype=np.complex128); x[0::2, 0] = u
    Hx = KP.apply_H_k(ref, nq, v0, kv, x)
    lam = (np.vdot(x, Hx) / np.vdot(x, x)).real
    want = 0.5 * np.sum((kv + Gv) ** 2); wrong = 0.5 * np.sum((kv - Gv) ** 2)
    assert abs(lam - want) < 1e-5 * want and abs(lam - wrong) > 0.1 * want
    assert np.linalg.norm(Hx - want * x) < 1e-3 * want * np.linalg.norm(x)


def test_conjugation_symmetry_k_to_minus_k():
    """B_y = 0, Delta real (the SOC-off twin): every table of H^k is real except -i k.G and the Bloch phases, so
    H^{-k} with P^{-k} = conj(P^k) is the complex conjugate of H^k."""
    cfg, ref0, refp, s = _ctx(natoms=1)
    assert np.abs(s.delta_soc_off.imag).max() == 0.0
    nq = 4; vq = _fields(ref0, nq, by=False); kv = np.array([0.2, 0.3, -0.1])
    pk = synth.bloch_pvals(s, ref0.node_coords(), kv)
    assert np.allclose(synth.bloch_pvals(s, ref0.node_coords(), -kv), pk.conj())
    X = synth.random_block(np.random.default_rng(6), 2 * ref0.M, 2)
    a = KP.apply_H_k(ref0, nq, vq, -kv, X.conj(), _proj(s, pk.conj(), s.delta_soc_off))
    b = KP.apply_H_k(ref0, nq, vq, kv, X, _proj(s, pk, s.delta_soc_off))
    assert np.allclose(a, b.conj(), atol=1e-12 * np.abs(b).max())


def test_chebyshev_filter_on_the_eigenbasis():
    """T_m of the dense matrix through its eigen-decomposition (numpy's chebval) against the recurrence."""
    cfg, ref0, refp, s = _ctx(ncell=(2, 2, 2), order=2, natoms=1)
    nq = 4; vq = _fields(ref0, nq); kv = (0.3, 0.1, -0.2)
    pk = synth.bloch_pvals(s, ref0.node_coords(), kv)
    apply = lambda Z: KP.apply_H_k(ref0, nq, vq, kv, Z, _proj(s, pk))
    n = 2 * ref0.M
    H = apply(np.eye(n, dtype=np.complex128))
    assert np.allclose(H, H.conj().T, atol=1e-11 * np.abs(H).max())
    lam, V = np.linalg.eigh(0.5 * (H + H.conj().T))
    a, b = lam[0] + 0.3 * (lam[-1] - lam[0]), lam[-1] + 0.05
    X = synth.random_block(np.random.default_rng(8), n, 3)
    for m in (0, 1, 2, 7):
        c = np.zeros(m + 1); c[m] = 1.0
        tm = np.polynomial.chebyshev.chebval((lam - 0.5 * (a + b)) / (0.5 * (b - a)), c)
        want = V @ (tm[:, None] * (V.conj().T @ X))
        got = KP.chebyshev_filter(apply, X, m, a, b)
        assert np.allclose(got, want, atol=1e-10 * np.abs(want).max())

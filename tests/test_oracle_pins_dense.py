"""Pins for oracle/dense_oracle.py (general-quadrature potential, dense cell-matrix apply; eq.79-84)."""
import itertools

import numpy as np
import pytest

from oracle import dense_oracle as D
from oracle import oracle as O
from paper_2410_02754_b200 import synth
from test_oracle_pins import _su2


def _ctx(ncell=(2, 2, 2), box=(2.0, 2.6, 1.8), order=3, bc=(0, 0, 0), natoms=0, seed=5):
    cfg = synth.Config(9, "gq", ncell, box, order, bc, natoms, "uniform", 4, 4, 0, seed)
    ref = O.RefCtx(cfg.ncell, cfg.box, cfg.order, cfg.bc)
    s = synth.make_system(cfg, ref.node_coords(), ref.mass_diag(), with_projectors=natoms > 0)
    ref.set_potential(np.zeros(ref.M), None)
    if natoms:
        ref.set_projectors(s.node_ptr, s.node_idx, s.nproj, s.pvals, s.atom_type, s.delta, s.delta_ptr)
    return cfg, ref, s


@pytest.mark.parametrize("p", [1, 2, 3, 5])
def test_lagrange_basis_at_points(p):
    xi, _ = O.gll(p)
    L = D.lagrange_at(p, xi)
    assert np.allclose(L, np.eye(p + 1), atol=1e-13)                      # nodal: l_i(xi_j) = delta_ij
    x = np.linspace(-1, 1, 7)
    L = D.lagrange_at(p, x)
    assert np.allclose(L.sum(0), 1.0, atol=1e-13)                         # partition of unity
    for k in range(p + 1):                                                # reproduces polynomials up to degree p
        assert np.allclose((xi ** k) @ L, x ** k, atol=1e-12)


def test_constant_potential_gives_the_consistent_mass_matrix():
    """v = c: V^(e) = c int N_a N_b = c (h/2)^3 Mhat (x) Mhat (x) Mhat with the exact 1-D mass matrix (closed form pinned in
    test_oracle_pins.py), provided n_q >= p + 1; its row sums are c times the cell's share of the lumped mass."""
    cfg, ref, _ = _ctx(order=3)
    nq = 5
    vq = np.zeros((ref.E, nq ** 3, 4)); vq[:, :, 0] = 1.7
    Vm = D.cell_potential_matrices(ref, nq, vq)
    _, Mh, _ = O.ref1d(3)
    h = [ref.box[d] / ref.ncell[d] for d in range(3)]
    want = 1.7 * np.kron(Mh * h[2] / 2, np.kron(Mh * h[1] / 2, Mh * h[0] / 2))
    assert np.allclose(Vm[0, 0], want, atol=1e-13 * np.abs(want).max())
    assert np.allclose(Vm[3, 0], want, atol=1e-13 * np.abs(want).max()) and np.abs(Vm[:, 1:]).max() == 0.0
    xi, w = O.gll(3)
    cellmass = np.einsum("c,b,a->cba", w * h[2] / 2, w * h[1] / 2, w * h[0] / 2).reshape(-1)
    assert np.allclose(Vm[0, 0].sum(1), 1.7 * cellmass, atol=1e-13)


def test_polynomial_potential_is_integrated_exactly_and_not_beyond():
    """One cell [0, hx] x [0, hy] x [0, hz]: u^T V w = int u w v for monomials; with v of degree s per direction the integrand has
    degree 2p + s per direction: exact iff 2 n_q - 1 >= 2p + s."""
    p = 2
    ref = O.RefCtx((1, 1, 1), (1.3, 0.9, 1.1), p, (2, 2, 2))        # free boundary: all 27 nodes of the cell kept
    coords = ref.node_coords(); conn = ref.connectivity()[0]
    s = 3
    for nq, exact in [(4, True), (3, False)]:
        pts = D.quadrature_points(ref, nq)
        vq = np.zeros((1, nq ** 3, 4))
        vq[0, :, 0] = pts[0, :, 0] ** s * pts[0, :, 1] ** s * pts[0, :, 2] ** s
        Vm = D.cell_potential_matrices(ref, nq, vq)[0, 0]
        worst = 0.0
        for (a, b, c), (d, e, f) in itertools.product([(0, 0, 0), (2, 1, 0), (1, 2, 2), (2, 2, 2)], repeat=2):
            u = np.zeros(27); w = np.zeros(27)
            u[:] = coords[conn, 0] ** a * coords[conn, 1] ** b * coords[conn, 2] ** c
            w[:] = coords[conn, 0] ** d * coords[conn, 1] ** e * coords[conn, 2] ** f
            got = u @ Vm @ w
            want = np.prod([L ** (k + 1) / (k + 1) for L, k in zip(ref.box, (a + d + s, b + e + s, c + f + s))])
            worst = max(worst, abs(got - want) / abs(want))
        assert (worst < 1e-12) if exact else (worst > 1e-6)


def test_apply_H_gq_hermitian_and_su2_and_limit():
    cfg, ref, s = _ctx(ncell=(2, 2, 2), order=3, natoms=1)
    nq = 5
    pts = D.quadrature_points(ref, nq)
    # smooth analytic fields at the quadrature points (periodic in the box)
    k = [2 * np.pi / L for L in ref.box]
    ph = pts[..., 0] * k[0] + 2 * pts[..., 1] * k[1] - pts[..., 2] * k[2]
    vq = np.stack([-1.0 + 0.3 * np.cos(ph), 0.2 * np.sin(ph), 0.1 * np.cos(2 * ph), 0.15 + 0.05 * np.sin(ph)], axis=-1)
    rng = np.random.default_rng(2)
    X = synth.random_block(rng, 2 * ref.M, 3); Yv = synth.random_block(rng, 2 * ref.M, 3)
    HX = D.apply_H_gq(ref, nq, vq, X); HY = D.apply_H_gq(ref, nq, vq, Yv)
    assert np.allclose(np.einsum("ij,ij->j", X.conj(), HY), np.einsum("ij,ij->j", Yv.conj(), HX).conj(), rtol=1e-12)     # Hermitian (B_y is the imaginary part)
    # SU(2): rotating B at the quadrature points by R and the spinors by U commutes with H (no SOC: Delta spin-diagonal)
    ref.set_projectors(s.node_ptr, s.node_idx, s.nproj, s.pvals, s.atom_type, s.delta_soc_off, s.delta_ptr)
    U, R = _su2(0.7, (0.5, -0.2, 0.6)); M = ref.M
    rot = lambda Z: (Z.reshape(M, 2, -1).transpose(0, 2, 1) @ U.T).transpose(0, 2, 1).reshape(2 * M, -1)
    vr = vq.copy(); vr[..., 1:] = vq[..., 1:] @ R.T
    assert np.allclose(D.apply_H_gq(ref, nq, vr, rot(X)), rot(D.apply_H_gq(ref, nq, vq, X)), atol=1e-12 * np.abs(HX).max())
    # linear in the fields; zero fields = the kinetic + nonlocal operator of the C oracle
    assert np.allclose(D.apply_H_gq(ref, nq, 0 * vq, X), ref.apply_H(X), atol=1e-13)
    # a uniform V shifts <x, H x> by V |x|^2-weighted consistent-mass form: here the weaker, exact statement sum_ab V_ab = V * volume
    vq2 = np.zeros_like(vq); vq2[..., 0] = 0.9
    assert abs(D.cell_potential_matrices(ref, nq, vq2)[:, 0].sum() - 0.9 * np.prod(ref.box)) < 1e-11

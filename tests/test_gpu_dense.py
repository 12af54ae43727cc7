"""GPU parity for SURVEY 8(f) NEXT-3: csf_quadrature_points / csf_set_potential_quadrature / csf_apply_H_dense (through
the C ABI) against oracle/dense_oracle.py (eq.79-84), element by element on the same seeded inputs.

Tolerance: relative Frobenius error <= 1e-11 and per-column maximum <= 1e-10, as for csf_apply_H (test_gpu_parity.py).
"""
import numpy as np
import pytest

from paper_2410_02754_b200 import synth, binding
from helpers import assert_block_close

pytestmark = pytest.mark.gpu
TOL = 1e-11


def _setup(ncell, box, order, bc, natoms, seed=11):
    from oracle import oracle as O
    cfg = synth.Config(9, "gq", tuple(ncell), tuple(box), order, tuple(bc), natoms, "uniform", 4, 4, 0, seed)
    ref = O.RefCtx(cfg.ncell, cfg.box, cfg.order, cfg.bc)
    s = synth.make_system(cfg, ref.node_coords(), ref.mass_diag(), with_projectors=natoms > 0)
    gpu = binding.Csf(cfg.ncell, cfg.box, cfg.order, cfg.bc)
    ref.set_potential(np.zeros(ref.M), None)           # the oracle's nodal potential is zero: apply_H_gq adds the quadrature part
    if natoms:
        for ctx in (ref, gpu):
            ctx.set_projectors(s.node_ptr, s.node_idx, s.nproj, s.pvals, s.atom_type, s.delta, s.delta_ptr)
    return ref, gpu, s


def _fields(pts, box, rng):
    """Smooth, box-periodic V_eff and B at the quadrature points (not polynomials of low degree: the rule matters)."""
    k = [2 * np.pi / b for b in box]
    x, y, z = pts[..., 0], pts[..., 1], pts[..., 2]
    a = rng.uniform(0.3, 1.0, size=8)
    vq = np.empty(pts.shape[:2] + (4,))
    vq[..., 0] = -1.5 + a[0] * np.cos(k[0] * x) * np.sin(k[1] * y + 0.3) + a[1] * np.cos(2 * k[2] * z)
    vq[..., 1] = 0.3 * a[2] * np.sin(k[0] * x + k[2] * z)
    vq[..., 2] = 0.3 * a[3] * np.cos(k[1] * y) * np.cos(k[0] * x + 0.7)
    vq[..., 3] = 0.3 * a[4] * np.sin(k[2] * z + k[1] * y) + 0.1 * a[5]
    return vq


def _gpu_apply_dense(gpu, X, ld=None):
    import torch
    nvec = X.shape[1]; ld = ld or nvec
    dX = torch.zeros((X.shape[0], ld), dtype=torch.complex128, device="cuda"); dX[:, :nvec] = torch.from_numpy(X).cuda()
    dX0 = dX.clone()
    dY = torch.full((X.shape[0], ld), 7.0 + 3.0j, dtype=torch.complex128, device="cuda")
    work = torch.empty(max(gpu.dense_workspace_bytes(nvec), 16), dtype=torch.uint8, device="cuda")
    gpu.apply_H_dense(dX, dY, ld, nvec, work)
    torch.cuda.synchronize()
    assert torch.equal(dX, dX0), "X was modified"
    out = dY.cpu().numpy()
    if ld > nvec:
        assert np.all(out[:, nvec:] == 7.0 + 3.0j), "padding columns were touched"
    return out[:, :nvec].copy()


@pytest.mark.parametrize("order,nq", [(1, 2), (2, 3), (3, 5), (4, 5), (5, 6), (5, 8)])
def test_quadrature_points_match_oracle(order, nq):
    from oracle import dense_oracle as D
    ref, gpu, _ = _setup((2, 3, 2), (2.0, 3.3, 1.8), order, (0, 1, 0), 0)
    assert np.allclose(gpu.quadrature_points(nq), D.quadrature_points(ref, nq), atol=1e-13)


@pytest.mark.parametrize("order,nq,natoms,nvec,ld", [(1, 2, 0, 5, 5), (2, 4, 0, 9, 12), (3, 5, 2, 7, 7), (4, 6, 2, 19, 19), (5, 7, 2, 10, 16), (6, 8, 0, 3, 3)])
@pytest.mark.parametrize("bc", [(0, 0, 0), (0, 1, 1)])
def test_apply_H_dense_against_oracle(order, nq, natoms, nvec, ld, bc):
    from oracle import dense_oracle as D
    ncell, box = ((3, 2, 3), (4.5, 3.2, 4.8)) if order <= 4 else ((2, 2, 3), (3.4, 3.6, 5.1))
    if natoms and order <= 3:
        ncell, box = (5, 5, 5), (7.5, 7.5, 7.5)
    ref, gpu, s = _setup(ncell, box, order, bc, natoms)
    vq = _fields(D.quadrature_points(ref, nq), box, s.rng)
    gpu.set_potential_quadrature(nq, vq)
    X = synth.random_block(s.rng, 2 * ref.M, nvec)
    assert_block_close(_gpu_apply_dense(gpu, X, ld=ld), D.apply_H_gq(ref, nq, vq, X), TOL)


def test_dense_path_with_the_nodal_rule_reproduces_apply_H():
    """Fields of low polynomial degree are integrated exactly by both rules only in special cases; a CONSTANT potential with
    n_q >= p + 1 gives the consistent mass matrix (dense), the nodal path the lumped one: they differ. What must agree exactly
    is the kinetic + nonlocal part: V = 0 on both paths."""
    from oracle import dense_oracle as D
    ref, gpu, s = _setup((3, 3, 3), (6.0, 6.0, 6.0), 3, (0, 0, 0), 2)
    nq = 4
    gpu.set_potential(np.zeros(ref.M), None)
    gpu.set_potential_quadrature(nq, np.zeros((ref.E, nq ** 3, 4)))
    X = synth.random_block(s.rng, 2 * ref.M, 6)
    import torch
    from helpers import gpu_apply_H
    Yd = _gpu_apply_dense(gpu, X)
    assert_block_close(Yd, gpu_apply_H(gpu, X), TOL)
    assert_block_close(Yd, ref.apply_H(X), TOL)


def test_single_periodic_cell_and_replacing_the_potential():
    """One cell per periodic direction (both end nodes of the cell are the same global node); the matrices are rebuilt when
    the potential is set again with another rule."""
    from oracle import dense_oracle as D
    ref, gpu, s = _setup((1, 2, 1), (1.6, 3.0, 1.4), 4, (0, 0, 0), 0)
    X = synth.random_block(s.rng, 2 * ref.M, 4)
    for nq in (5, 7):
        vq = _fields(D.quadrature_points(ref, nq), (1.6, 3.0, 1.4), s.rng)
        gpu.set_potential_quadrature(nq, vq)
        assert_block_close(_gpu_apply_dense(gpu, X), D.apply_H_gq(ref, nq, vq, X), TOL)


def test_dense_argument_errors():
    import torch
    ref, gpu, s = _setup((2, 2, 2), (2.0, 2.0, 2.0), 2, (0, 0, 0), 0)
    X = torch.zeros((2 * ref.M, 4), dtype=torch.complex128, device="cuda"); Y = torch.zeros_like(X)
    with pytest.raises(binding.CsfError) as ei:
        gpu.apply_H_dense(X, Y, 4, 4)
    assert ei.value.code == binding.CSF_ESTATE
    with pytest.raises(binding.CsfError) as ei:
        gpu.quadrature_points(17)
    assert ei.value.code == binding.CSF_EINVAL
    gpu.set_potential_quadrature(3, np.zeros((ref.E, 27, 4)))
    with pytest.raises(binding.CsfError) as ei:
        gpu.apply_H_dense(X, X, 4, 4)
    assert ei.value.code == binding.CSF_EINVAL
    gpu.apply_H_dense(X, Y, 4, 0)                       # nvec = 0: no-op

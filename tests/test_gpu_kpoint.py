"""GPU parity for SURVEY 8(f) NEXT-2: the k-point Hamiltonian with complex projectors on the dense path (csf_set_kpoint,
csf_set_projectors_complex, csf_apply_H_dense, csf_filter_dense; through the C ABI) against oracle/kpoint_oracle.py
(eq.21-24, eq.40-42, eq.70), element by element on the same seeded inputs.

Tolerance: relative Frobenius error <= 1e-11, per-column maximum <= 1e-10 (as test_gpu_parity.py).
"""
import numpy as np
import pytest

from paper_2410_02754_b200 import synth, binding
from helpers import assert_block_close, gpu_filter

pytestmark = pytest.mark.gpu
TOL = 1e-11


def _setup(ncell, box, order, bc, natoms, kvec, nq, seed=21, cplx=True):
    from oracle import oracle as O
    from oracle import dense_oracle as D
    cfg = synth.Config(9, "kp", tuple(ncell), tuple(box), order, tuple(bc), natoms, "uniform", 4, 4, 0, seed)
    ref0 = O.RefCtx(cfg.ncell, cfg.box, cfg.order, cfg.bc)
    ref0.set_potential(np.zeros(ref0.M), None)
    s = synth.make_system(cfg, ref0.node_coords(), ref0.mass_diag(), with_projectors=natoms > 0)
    gpu = binding.Csf(cfg.ncell, cfg.box, cfg.order, cfg.bc)
    proj = None
    if natoms:
        pk = synth.bloch_pvals(s, ref0.node_coords(), kvec) if cplx else s.pvals.astype(np.complex128)
        proj = (s.node_ptr, s.node_idx, s.nproj, pk, s.atom_type, s.delta, s.delta_ptr)
        if cplx:
            gpu.set_projectors_complex(*proj)
        else:
            gpu.set_projectors(s.node_ptr, s.node_idx, s.nproj, s.pvals, s.atom_type, s.delta, s.delta_ptr)
    pts = D.quadrature_points(ref0, nq)
    kk = [2 * np.pi / b for b in box]
    ph = pts[..., 0] * kk[0] - pts[..., 1] * kk[1] + 2 * pts[..., 2] * kk[2]
    vq = np.stack([-1.2 + 0.4 * np.cos(ph), 0.2 * np.sin(ph), 0.15 * np.cos(2 * ph), 0.1 + 0.05 * np.sin(ph)], axis=-1)
    gpu.set_kpoint(kvec)
    gpu.set_potential_quadrature(nq, vq)
    return ref0, gpu, s, vq, proj


def _dense(gpu, X, ld=None, filt=None):
    import torch
    nvec = X.shape[1]; ld = ld or nvec
    dX = torch.zeros((X.shape[0], ld), dtype=torch.complex128, device="cuda"); dX[:, :nvec] = torch.from_numpy(X).cuda()
    dX0 = dX.clone()
    dY = torch.full((X.shape[0], ld), 7.0 + 3.0j, dtype=torch.complex128, device="cuda")
    work = torch.empty(max(gpu.dense_workspace_bytes(nvec), 16), dtype=torch.uint8, device="cuda")
    if filt is None:
        gpu.apply_H_dense(dX, dY, ld, nvec, work)
    else:
        gpu.filter_dense(dX, dY, ld, nvec, filt[0], filt[1], filt[2], work)
    torch.cuda.synchronize()
    assert torch.equal(dX, dX0), "X was modified"
    out = dY.cpu().numpy()
    if ld > nvec:
        assert np.all(out[:, nvec:] == 7.0 + 3.0j), "padding columns were touched"
    return out[:, :nvec].copy()


@pytest.mark.parametrize("order,nq,natoms,nvec,ld,bc", [(2, 4, 0, 5, 5, (0, 0, 0)), (3, 5, 2, 9, 12, (0, 0, 0)), (4, 6, 2, 19, 19, (0, 0, 1)),
                                                         (5, 7, 2, 10, 16, (0, 0, 0)), (6, 8, 0, 3, 3, (0, 1, 0))])
def test_apply_H_k_against_oracle(order, nq, natoms, nvec, ld, bc):
    from oracle import kpoint_oracle as KP
    ncell, box = ((3, 2, 3), (4.5, 3.2, 4.8)) if order <= 4 else ((2, 2, 3), (3.4, 3.6, 5.1))
    if natoms and order <= 3:
        ncell, box = (5, 5, 5), (7.5, 7.5, 7.5)
    kvec = np.array([0.37, -0.21, 0.13])
    ref0, gpu, s, vq, proj = _setup(ncell, box, order, bc, natoms, kvec, nq)
    X = synth.random_block(s.rng, 2 * ref0.M, nvec)
    assert_block_close(_dense(gpu, X, ld=ld), KP.apply_H_k(ref0, nq, vq, kvec, X, proj), TOL)


@pytest.mark.parametrize("degree", [0, 1, 2, 5, 8])
@pytest.mark.parametrize("kvec", [(0.0, 0.0, 0.0), (0.25, 0.1, -0.3)])
def test_filter_dense_against_oracle(degree, kvec):
    from oracle import kpoint_oracle as KP
    kvec = np.array(kvec)
    ref0, gpu, s, vq, proj = _setup((5, 5, 5), (7.5, 7.5, 7.5), 3, (0, 0, 0), 2, kvec, 5)
    X = synth.random_block(s.rng, 2 * ref0.M, 6)
    a, b = 4.0, 31.0                          # an interval inside the spectrum: the filter amplifies what lies below a
    want = KP.chebyshev_filter(lambda Z: KP.apply_H_k(ref0, 5, vq, kvec, Z, proj), X, degree, a, b)
    assert_block_close(_dense(gpu, X, ld=8, filt=(degree, a, b)), want, TOL)


def test_filter_dense_agrees_with_the_sum_factorised_filter_where_both_apply():
    """Zero potential, Gamma point, real projectors: the two GPU filters hold the same operator."""
    ref0, gpu, s, vq, proj = _setup((3, 3, 3), (6.0, 6.0, 6.0), 4, (0, 0, 0), 2, np.zeros(3), 5, cplx=False)
    gpu.set_potential(np.zeros(ref0.M), None)
    gpu.set_potential_quadrature(5, np.zeros_like(vq))
    X = synth.random_block(s.rng, 2 * ref0.M, 9)
    a, b = 3.0, 40.0
    assert_block_close(_dense(gpu, X, filt=(6, a, b)), gpu_filter(gpu, X, 6, a, b), TOL)


def test_state_rules_of_the_kpoint_calls():
    import torch
    kvec = np.array([0.2, 0.0, -0.1])
    ref0, gpu, s, vq, proj = _setup((3, 3, 3), (6.0, 6.0, 6.0), 3, (0, 0, 0), 2, kvec, 4)
    gpu.set_potential(np.zeros(ref0.M), None)
    X = torch.zeros((2 * ref0.M, 4), dtype=torch.complex128, device="cuda"); Y = torch.zeros_like(X)
    work = torch.empty(max(gpu.workspace_bytes(4), gpu.dense_workspace_bytes(4)), dtype=torch.uint8, device="cuda")
    # the sum-factorised entry points refuse while a k-point / complex projectors are set
    for call in (lambda: gpu.apply_H(X, Y, 4, 4, work), lambda: gpu.filter(X, Y, 4, 4, 3, 1.0, 9.0, 0, work), lambda: gpu.apply_H_static(X, Y, 4, 4)):
        with pytest.raises(binding.CsfError) as ei:
            call()
        assert ei.value.code == binding.CSF_ESTATE and "dense path" in str(ei.value)
    # a new k-point invalidates the cell matrices
    gpu.set_kpoint((0.0, 0.0, 0.0))
    with pytest.raises(binding.CsfError) as ei:
        gpu.apply_H_dense(X, Y, 4, 4, work)
    assert ei.value.code == binding.CSF_ESTATE
    # back to the Gamma point with real projectors: everything is served again
    gpu.set_projectors(s.node_ptr, s.node_idx, s.nproj, s.pvals, s.atom_type, s.delta, s.delta_ptr)
    gpu.set_potential_quadrature(4, vq)
    gpu.apply_H(X, Y, 4, 4, work); gpu.apply_H_dense(X, Y, 4, 4, work)
    torch.cuda.synchronize()


def test_rayleigh_ritz_and_lanczos_at_a_kpoint():
    """csf_rr_project and csf_lanczos apply the operator the context holds: Hhat^k on the dense path here."""
    import torch
    from oracle import kpoint_oracle as KP
    from oracle import subspace_oracle as S
    from helpers import rel_fro
    kvec = np.array([0.3, -0.2, 0.15])
    ref0, gpu, s, vq, proj = _setup((5, 5, 5), (7.5, 7.5, 7.5), 3, (0, 0, 0), 2, kvec, 5)
    apply = lambda Z: KP.apply_H_k(ref0, 5, vq, kvec, Z, proj)
    N = 12
    X = synth.random_block(s.rng, 2 * ref0.M, N)
    dX = torch.from_numpy(X).cuda()
    dHs = torch.empty((N, N), dtype=torch.complex128, device="cuda"); dSs = torch.empty_like(dHs); dQ = torch.empty_like(dHs)
    work = torch.empty(gpu.rr_workspace_bytes(N), dtype=torch.uint8, device="cuda")
    gpu.rr_project(dX, N, N, dHs, dSs, work)
    torch.cuda.synchronize()
    Hr, Sr = S.rr_project(apply, X)
    assert rel_fro(dHs.cpu().numpy(), Hr) < 1e-11 and rel_fro(dSs.cpu().numpy(), Sr) < 1e-12
    lam = gpu.rr_solve(dHs, dSs, N, dQ)
    lam_ref, _ = S.rr_solve(Hr, Sr)
    assert np.allclose(lam, lam_ref, rtol=0, atol=1e-9 * np.abs(lam_ref).max())
    v0 = synth.random_block(s.rng, 2 * ref0.M, 1)
    lw = torch.empty(gpu.lanczos_workspace_bytes(), dtype=torch.uint8, device="cuda")
    al, be = gpu.lanczos(torch.from_numpy(v0).cuda(), 12, lw)
    alr, ber = S.lanczos(apply, v0, 12)
    assert np.allclose(al[:8], alr[:8], rtol=1e-10) and np.allclose(be[:8], ber[:8], rtol=1e-10)


def test_bench_launch_configuration_on_sampled_columns():
    """The launch configuration bench.py's dense leg times (order 5, cells of 1 bohr, 256 vectors = 16 chunks of 16 per cell, n_q = 8,
    atoms with 18 projectors) on a 6^3-cell mesh, at a k-point with complex projectors: one H apply and a degree-6 filter of the whole
    block on the GPU, the columns {0..3, 252..255} against the oracle."""
    import torch
    from oracle import kpoint_oracle as KP
    from oracle import oracle as O
    from oracle import dense_oracle as D
    cfg = synth.scaled_config(synth.CONFIGS[3], (6, 6, 6), 4, nvec=256)
    ref0 = O.RefCtx(cfg.ncell, cfg.box, cfg.order, cfg.bc); ref0.set_potential(np.zeros(ref0.M), None)
    s = synth.make_system(cfg, ref0.node_coords(), ref0.mass_diag())
    kvec = np.array([0.21, -0.13, 0.08]); nq = 8
    pk = synth.bloch_pvals(s, ref0.node_coords(), kvec)
    proj = (s.node_ptr, s.node_idx, s.nproj, pk, s.atom_type, s.delta, s.delta_ptr)
    pts = D.quadrature_points(ref0, nq)
    kk = [2 * np.pi / b for b in cfg.box]
    vq = np.empty(pts.shape[:2] + (4,))
    vq[..., 0] = -1.0 + 0.5 * np.cos(kk[0] * pts[..., 0]) * np.cos(kk[1] * pts[..., 1]) * np.cos(kk[2] * pts[..., 2])
    vq[..., 1] = 0.1 * np.sin(kk[0] * pts[..., 0]); vq[..., 2] = 0.1 * np.sin(kk[1] * pts[..., 1]); vq[..., 3] = 0.1 * np.cos(kk[2] * pts[..., 2])
    gpu = binding.Csf(cfg.ncell, cfg.box, cfg.order, cfg.bc)
    gpu.set_projectors_complex(*proj); gpu.set_kpoint(kvec); gpu.set_potential_quadrature(nq, vq)
    N = cfg.nvec
    X = synth.random_block(s.rng, 2 * ref0.M, N)
    cols = [0, 1, 2, 3, N - 4, N - 3, N - 2, N - 1]
    apply = lambda Z: KP.apply_H_k(ref0, nq, vq, kvec, Z, proj)
    assert_block_close(_dense(gpu, X)[:, cols], apply(X[:, cols]), TOL)
    a, b = 6.0, 140.0
    assert_block_close(_dense(gpu, X, filt=(6, a, b))[:, cols], KP.chebyshev_filter(apply, X[:, cols], 6, a, b), TOL)

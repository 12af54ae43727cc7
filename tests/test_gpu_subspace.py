"""GPU parity of the subspace steps around the filter (SURVEY 8(f) NEXT-1 Rayleigh-Ritz, NEXT-4 density / magnetisation and
Lanczos) against oracle/subspace_oracle.py, through the C ABI. Tolerances: 1e-11 relative Frobenius for the projected
matrices and the rotated block (sums over all 2M rows in FP64), 1e-9 on Ritz values (conditioning of the pencil)."""
import numpy as np
import pytest

from paper_2410_02754_b200 import synth, bounds
from helpers import setup_pair, rel_fro, assert_block_close

pytestmark = pytest.mark.gpu


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _case(name):
    if name == "cfg0":
        return synth.CONFIGS[0], 16
    if name == "p5_slab":
        return synth.scaled_config(synth.CONFIGS[2], (3, 3, 4), 3, nvec=24, degree=6), 24        # 2N = 48 < one tile
    if name == "p4_bulk":
        return synth.scaled_config(synth.CONFIGS[4], (6, 6, 6), 4, nvec=40, degree=6), 40        # 2N = 80: one full and one ragged tile
    return synth.scaled_config(synth.CONFIGS[3], (5, 5, 5), 4, nvec=72, degree=6), 72            # 2N = 144: three tile columns


@pytest.mark.parametrize("case", ["cfg0", "p5_slab", "p4_bulk", "p5_bulk72"])
def test_rr_project_solve_rotate(case):
    import torch
    from oracle import subspace_oracle as S
    cfg, N = _case(case)
    ref, gpu, s = setup_pair(cfg)
    X = synth.random_block(s.rng, 2 * ref.M, N)
    ld = N + 3
    dX = torch.zeros((2 * ref.M, ld), dtype=torch.complex128, device="cuda"); dX[:, :N] = _dev(X)
    dHs = torch.empty((N, N), dtype=torch.complex128, device="cuda"); dSs = torch.empty_like(dHs); dQ = torch.empty_like(dHs)
    work = torch.empty(gpu.rr_workspace_bytes(N), dtype=torch.uint8, device="cuda")
    gpu.rr_project(dX, ld, N, dHs, dSs, work)
    torch.cuda.synchronize()
    Hs, Ss = dHs.cpu().numpy(), dSs.cpu().numpy()
    Hr, Sr = S.rr_project(ref.apply_H, X)
    assert rel_fro(Hs, Hr) < 1e-11 and rel_fro(Ss, Sr) < 1e-12
    assert np.array_equal(Hs, Hs.conj().T) and np.array_equal(Ss, Ss.conj().T)          # exactly Hermitian
    lam = gpu.rr_solve(dHs, dSs, N, dQ)
    Q = dQ.cpu().numpy()
    lam_ref, _ = S.rr_solve(Hr, Sr)
    assert np.allclose(lam, lam_ref, rtol=0, atol=1e-9 * np.abs(lam_ref).max())
    assert np.allclose(Q.conj().T @ Ss @ Q, np.eye(N), atol=1e-10)
    assert np.linalg.norm(Hs @ Q - Ss @ Q * lam) < 1e-9 * np.linalg.norm(Hs)
    ldu = N + 1
    dU = torch.full((2 * ref.M, ldu), 7.0 + 3.0j, dtype=torch.complex128, device="cuda")
    gpu.rr_rotate(dX, ld, N, dQ, dU, ldu, work)
    torch.cuda.synchronize()
    U = dU.cpu().numpy()
    assert np.all(U[:, N:] == 7.0 + 3.0j), "padding columns were touched"
    assert_block_close(U[:, :N], S.rr_rotate(X, Q), 1e-12)
    # the rotated block diagonalises Hhat in the subspace (eq.72)
    assert np.allclose(U[:, :N].conj().T @ ref.apply_H(U[:, :N]), np.diag(lam), atol=1e-8 * np.abs(lam).max())
    assert torch.equal(dX[:, :N].cpu(), torch.from_numpy(X)), "X was modified"


def test_chfsi_pass_on_gpu_matches_oracle(cfg0_oracle):
    """filter -> project -> solve -> rotate on the GPU against the same pass on the oracle: same Ritz values, same subspace."""
    import torch
    from oracle import subspace_oracle as S
    ref, a, b, X = (cfg0_oracle[k] for k in ("ctx", "a", "b", "X"))
    _, gpu, _ = setup_pair(synth.CONFIGS[0])
    N = X.shape[1]
    dX = _dev(X); dY = torch.empty_like(dX); dU = torch.empty_like(dX)
    dHs = torch.empty((N, N), dtype=torch.complex128, device="cuda"); dSs = torch.empty_like(dHs); dQ = torch.empty_like(dHs)
    work = torch.empty(max(gpu.workspace_bytes(N), gpu.rr_workspace_bytes(N)), dtype=torch.uint8, device="cuda")
    gpu.filter(dX, dY, N, N, 8, a, b, 0, work)
    gpu.rr_project(dY, N, N, dHs, dSs, work)
    lam = gpu.rr_solve(dHs, dSs, N, dQ)
    gpu.rr_rotate(dY, N, N, dQ, dU, N, work)
    torch.cuda.synchronize()
    Yr = ref.filter(X, 8, a, b)
    lam_ref, Qr = S.rr_solve(*S.rr_project(ref.apply_H, Yr))
    assert np.allclose(lam, lam_ref, atol=1e-8 * np.abs(lam_ref).max())
    U = dU.cpu().numpy(); Ur = S.rr_rotate(Yr, Qr)
    # same subspace, vector by vector up to a phase (non-degenerate Ritz values): |<u_i, ur_i>| = 1
    ov = np.abs(np.einsum("ij,ij->j", Ur.conj(), U))
    gaps = np.min(np.abs(np.subtract.outer(lam_ref, lam_ref)) + np.eye(N) * 1e9, axis=1)
    assert np.all(ov[gaps > 1e-3] > 1 - 1e-8)


@pytest.mark.parametrize("case", ["cfg0", "p5_slab"])
def test_density_and_magnetisation(case):
    import torch
    from oracle import subspace_oracle as S
    cfg, N = _case(case)
    ref, gpu, s = setup_pair(cfg, with_projectors=False)
    X = synth.random_block(s.rng, 2 * ref.M, N)
    occ = np.linspace(1.0, 0.05, N)
    ld = N + 2
    dX = torch.zeros((2 * ref.M, ld), dtype=torch.complex128, device="cuda"); dX[:, :N] = _dev(X)
    out = torch.full((ref.M, 4), 5.0, dtype=torch.float64, device="cuda")
    gpu.density(dX, ld, N, occ, out)
    torch.cuda.synchronize()
    rho, m = S.density(X, occ, ref.mass_diag())
    got = out.cpu().numpy()
    assert np.allclose(got[:, 0], rho, rtol=1e-12, atol=1e-14 * rho.max())
    assert np.allclose(got[:, 1:], m, rtol=0, atol=1e-12 * np.abs(rho).max())
    # blocks of states accumulate: two halves added = the whole
    h = N // 2
    out2 = torch.zeros_like(out)
    gpu.density(dX, ld, h, occ[:h], out2, accumulate=False)
    d2 = dX[:, h:].contiguous()
    gpu.density(d2, d2.shape[1], N - h, occ[h:], out2, accumulate=True)
    torch.cuda.synchronize()
    assert np.allclose(out2.cpu().numpy(), got, rtol=1e-12, atol=1e-13 * rho.max())


@pytest.mark.parametrize("case", ["cfg0", "p4_bulk"])
def test_lanczos_on_device(case):
    import torch
    from oracle import subspace_oracle as S
    from paper_2410_02754_b200 import binding
    cfg, _ = _case(case)
    ref, gpu, s = setup_pair(cfg)
    v0 = synth.random_block(s.rng, 2 * ref.M, 1) * 3.7          # any non-zero norm
    work = torch.empty(gpu.lanczos_workspace_bytes(), dtype=torch.uint8, device="cuda")
    al, be = gpu.lanczos(_dev(v0), 20, work)
    alr, ber = S.lanczos(ref.apply_H, v0, 20)
    assert len(al) == 20
    # the recurrence is sensitive to rounding in its late coefficients: the early ones agree closely, the Ritz extremes throughout
    assert np.allclose(al[:8], alr[:8], rtol=1e-10) and np.allclose(be[:8], ber[:8], rtol=1e-10)
    tmin, tmax = binding.tridiag_extremes(al, be)
    rmin, rmax = S.ritz_extremes(alr, ber)
    assert abs(tmin - rmin) < 1e-8 * abs(rmax) and abs(tmax - rmax) < 1e-8 * abs(rmax)
    # csf_tridiag_extremes against LAPACK on the same coefficients
    T = np.diag(al) + np.diag(be[:-1], 1) + np.diag(be[:-1], -1)
    th = np.linalg.eigvalsh(T)
    assert abs(tmin - th[0]) < 1e-12 * abs(th[-1]) and abs(tmax - th[-1]) < 1e-12 * abs(th[-1])
    # the bounds helper of the harness (host Lanczos through apply_H) and the device Lanczos give the same filter bounds from the same start
    assert tmax + be[-1] > rmax


def test_rr_at_full_size_config3():
    """Whole block of config 3 (N = 256): the 8 x 8 corner blocks of Hs and Ss against the oracle on the columns {0..3, B-4..B-1};
    sampled rows of U = X Q against NumPy; trace identities at full size."""
    import torch
    from oracle import oracle as O
    from oracle import subspace_oracle as S
    from paper_2410_02754_b200 import binding
    cfg = synth.CONFIGS[3]
    ref = O.RefCtx(cfg.ncell, cfg.box, cfg.order, cfg.bc)
    sysm = synth.make_system(cfg, ref.node_coords(), ref.mass_diag())
    gpu = binding.Csf(cfg.ncell, cfg.box, cfg.order, cfg.bc, stream=torch.cuda.current_stream().cuda_stream)
    for ctx in (ref, gpu):
        ctx.set_potential(sysm.veff, sysm.bxyz)
        ctx.set_projectors(sysm.node_ptr, sysm.node_idx, sysm.nproj, sysm.pvals, sysm.atom_type, sysm.delta, sysm.delta_ptr)
    N = cfg.nvec; rows = 2 * ref.M
    gen = torch.Generator(device="cuda"); gen.manual_seed(77)
    X = torch.empty((rows, N), dtype=torch.complex128, device="cuda")
    torch.view_as_real(X).normal_(0.0, np.sqrt(0.5), generator=gen)
    dHs = torch.empty((N, N), dtype=torch.complex128, device="cuda"); dSs = torch.empty_like(dHs); dQ = torch.empty_like(dHs)
    work = torch.empty(gpu.rr_workspace_bytes(N), dtype=torch.uint8, device="cuda")
    gpu.rr_project(X, N, N, dHs, dSs, work)
    torch.cuda.synchronize()
    cols = [0, 1, 2, 3, N - 4, N - 3, N - 2, N - 1]
    Xh = np.ascontiguousarray(X[:, cols].cpu().numpy())
    Hr, Sr = S.rr_project(ref.apply_H, Xh)
    Hs, Ss = dHs.cpu().numpy(), dSs.cpu().numpy()
    assert rel_fro(Hs[np.ix_(cols, cols)], Hr) < 1e-11 and rel_fro(Ss[np.ix_(cols, cols)], Sr) < 1e-12
    assert abs(np.trace(Ss).real - float((X.abs() ** 2).sum().item())) < 1e-11 * np.trace(Ss).real
    lam = gpu.rr_solve(dHs, dSs, N, dQ)
    assert np.all(np.diff(lam) >= 0)
    U = torch.empty_like(X)
    gpu.rr_rotate(X, N, N, dQ, U, N, work)
    torch.cuda.synchronize()
    pick = torch.tensor([0, 1, 12345, rows // 2, rows - 2, rows - 1], device="cuda")
    want = X[pick].cpu().numpy() @ dQ.cpu().numpy()
    assert rel_fro(U[pick].cpu().numpy(), want) < 1e-12
    # U^dagger U = I: the rotated block is orthonormal (one more projection, on U)
    del X
    gpu.rr_project(U, N, N, dHs, dSs, work)
    torch.cuda.synchronize()
    assert np.allclose(dSs.cpu().numpy(), np.eye(N), atol=1e-9)
    assert np.allclose(dHs.cpu().numpy(), np.diag(lam), atol=1e-7 * np.abs(lam).max())

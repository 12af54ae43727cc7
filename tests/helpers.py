"""Shared set-up for the GPU parity tests: the same seeded synthetic system on the oracle and on libcsf."""
import numpy as np

from paper_2410_02754_b200 import synth


def rel_fro(y, yref):
    return float(np.linalg.norm(y - yref) / max(np.linalg.norm(yref), 1e-300))


def col_err_max(y, yref):
    """Largest per-column relative 2-norm error (SURVEY 8(c) "also report the per-column maximum"): after Chebyshev
    amplification a wrong weakly-amplified column would hide under the strongly-amplified ones in the block norm."""
    num = np.linalg.norm(y - yref, axis=0); den = np.maximum(np.linalg.norm(yref, axis=0), 1e-300)
    return float((num / den).max())


def assert_block_close(y, yref, tol, col_tol=None):
    """Block Frobenius error < tol (BASELINE.json's metric) and every column on its own < col_tol (default 10 tol)."""
    e = rel_fro(y, yref); ec = col_err_max(y, yref)
    assert e < tol, f"relative Frobenius error {e:.3e} >= {tol:.1e}"
    assert ec < (col_tol if col_tol is not None else 10 * tol), f"per-column maximum error {ec:.3e}"
    return e, ec


def setup_pair(cfg, with_projectors=True, assemble_sparse=True, soc_off=False):
    """Returns (oracle ctx, gpu ctx, system). Inputs are generated once from the ORACLE's coordinates/masses;
    the GPU library's own coordinates and masses are asserted to agree in test_gpu_parity.py."""
    from oracle import oracle as O
    from paper_2410_02754_b200 import binding
    ref = O.RefCtx(cfg.ncell, cfg.box, cfg.order, cfg.bc, assemble_sparse=assemble_sparse)
    sysm = synth.make_system(cfg, ref.node_coords(), ref.mass_diag(), with_projectors=with_projectors)
    gpu = binding.Csf(cfg.ncell, cfg.box, cfg.order, cfg.bc)
    delta = sysm.delta_soc_off if soc_off else sysm.delta
    for ctx in (ref, gpu):
        ctx.set_potential(sysm.veff, sysm.bxyz)
        if with_projectors:
            ctx.set_projectors(sysm.node_ptr, sysm.node_idx, sysm.nproj, sysm.pvals, sysm.atom_type, delta, sysm.delta_ptr)
    return ref, gpu, sysm


def gpu_apply_H(gpu, X, ld=None):
    """X: host complex128 [2M, nvec] -> Hhat X through the C ABI (device buffers via torch)."""
    import torch
    nvec = X.shape[1]; ld = ld or nvec
    dX = torch.zeros((X.shape[0], ld), dtype=torch.complex128, device="cuda"); dX[:, :nvec] = torch.from_numpy(X).cuda()
    dY = torch.full((X.shape[0], ld), 7.0 + 3.0j, dtype=torch.complex128, device="cuda")
    wb = max(gpu.workspace_bytes(nvec), 16)
    work = torch.empty(wb, dtype=torch.uint8, device="cuda")
    gpu.apply_H(dX, dY, ld, nvec, work)
    torch.cuda.synchronize()
    out = dY.cpu().numpy()
    if ld > nvec:
        assert np.all(out[:, nvec:] == 7.0 + 3.0j), "padding columns were touched"
    return out[:, :nvec].copy()


def gpu_filter(gpu, X, degree, a, b, ld=None):
    import torch
    nvec = X.shape[1]; ld = ld or nvec
    dX = torch.zeros((X.shape[0], ld), dtype=torch.complex128, device="cuda"); dX[:, :nvec] = torch.from_numpy(X).cuda()
    dX0 = dX.clone()
    dY = torch.full((X.shape[0], ld), 7.0 + 3.0j, dtype=torch.complex128, device="cuda")
    work = torch.empty(max(gpu.workspace_bytes(nvec), 16), dtype=torch.uint8, device="cuda")
    gpu.filter(dX, dY, ld, nvec, degree, a, b, 0, work)
    torch.cuda.synchronize()
    assert torch.equal(dX, dX0), "X was modified"
    out = dY.cpu().numpy()
    if ld > nvec:
        assert np.all(out[:, nvec:] == 7.0 + 3.0j), "padding columns were touched"
    return out[:, :nvec].copy()

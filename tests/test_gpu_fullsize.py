"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (ld = nvec = the config's block).

config 1: the whole block against the oracle's filter. configs 2-4: the filter of the whole block, both modes, against
the oracle's filter on the 8 columns {0..3, B-4..B-1}; and, because the oracle cannot filter more columns in seconds,
  (a) sampled rows of Hhat X against the oracle's row-wise evaluation straight from the element definitions
      (`ref_apply_H_rows`, no global CSR), on columns copied back from the device block, with rows chosen on cell
      faces / edges / corners, on the periodic wrap, next to Dirichlet faces and inside projector supports;
  (b) properties that hold at any size, on the CUDA path alone: Hermiticity <x, H y> = conj <y, H x>, and the Chebyshev
      product identity 2 T_j T_k X = T_{j+k} X + T_{|j-k|} X (three library calls against each other).
Tolerance 1e-11 (relative Frobenius), as for the small cases.
"""
import numpy as np
import pytest

from paper_2410_02754_b200 import synth, bounds
from helpers import rel_fro, assert_block_close

pytestmark = pytest.mark.gpu
TOL = 1e-11


def _setup(cfg, sparse):
    import torch
    from oracle import oracle as O
    from paper_2410_02754_b200 import binding
    ref = O.RefCtx(cfg.ncell, cfg.box, cfg.order, cfg.bc, assemble_sparse=sparse)
    sysm = synth.make_system(cfg, ref.node_coords(), ref.mass_diag())
    gpu = binding.Csf(cfg.ncell, cfg.box, cfg.order, cfg.bc, stream=torch.cuda.current_stream().cuda_stream)
    for ctx in (ref, gpu):
        ctx.set_potential(sysm.veff, sysm.bxyz)
        ctx.set_projectors(sysm.node_ptr, sysm.node_idx, sysm.nproj, sysm.pvals, sysm.atom_type, sysm.delta, sysm.delta_ptr)
    return ref, gpu, sysm


def _device_block(rows, nvec, seed):
    import torch
    gen = torch.Generator(device="cuda"); gen.manual_seed(seed)
    X = torch.empty((rows, nvec), dtype=torch.complex128, device="cuda")
    torch.view_as_real(X).normal_(0.0, np.sqrt(0.5), generator=gen)
    return X


def test_config1_whole_block_filter():
    import torch
    cfg = synth.CONFIGS[1]
    ref, gpu, sysm = _setup(cfg, sparse=True)
    a, b, _, _ = bounds.lanczos_bounds(lambda v: ref.apply_H(v), 2 * ref.M)
    X = synth.random_block(sysm.rng, 2 * ref.M, cfg.nvec)
    dX = torch.from_numpy(X).cuda(); dY = torch.empty_like(dX)
    work = torch.empty(gpu.workspace_bytes(cfg.nvec), dtype=torch.uint8, device="cuda")
    gpu.filter(dX, dY, cfg.nvec, cfg.nvec, cfg.degree, a, b, 0, work)
    torch.cuda.synchronize()
    assert rel_fro(dY.cpu().numpy(), ref.filter(X, cfg.degree, a, b)) < TOL


def _sample_rows(cfg, sysm, rng, n_random=24):
    """Spinor rows 2I+alpha: structured picks (cell corners / edges / faces, first and last nodes = periodic wrap or
    next to a Dirichlet face), nodes inside projector supports, and random ones."""
    nx, ny, nz = cfg.nfree; p = cfg.order
    picks = []
    for gx, gy, gz in [(0, 0, 0), (nx - 1, ny - 1, nz - 1), (p, p, p), (p, 1, 2), (1, p, 2 * p), (nx - 1, 0, p), (0, ny - 1, nz - 1),
                       (2 * p, 3, nz - 1), (3, 2 * p, 0), (nx // 2, ny // 2, nz // 2), (p + 1, p + 2, p + 3), (nx - p, ny - p, nz - p)]:
        picks.append(gx % nx + nx * (gy % ny + ny * (gz % nz)))
    for gz in range(0, nz, 16 * p):          # z-planes where a 16-cell segment of the cell-per-iteration kernel hands over its face
        picks += [nx // 3 + nx * (ny // 3 + ny * gz), (2 * p) + nx * (p + ny * gz)]
    picks += [int(sysm.node_idx[int(t)]) for t in rng.integers(0, len(sysm.node_idx), 12)]
    picks += [int(i) for i in rng.integers(0, cfg.M, n_random)]
    rows = []
    for k, I in enumerate(picks):
        rows.append(2 * I + (k & 1))
    return np.unique(np.array(rows, dtype=np.int64))


@pytest.mark.parametrize("k", [2, 3, 4])
def test_sampled_rows_of_apply_H_at_full_size(k):
    import torch
    cfg = synth.CONFIGS[k]
    ref, gpu, sysm = _setup(cfg, sparse=False)
    rows_n = 2 * ref.M; nvec = cfg.nvec
    dX = _device_block(rows_n, nvec, 4242 + k); dY = torch.empty_like(dX)
    work = torch.empty(gpu.workspace_bytes(nvec), dtype=torch.uint8, device="cuda")
    gpu.apply_H(dX, dY, nvec, nvec, work)
    torch.cuda.synchronize()
    cols = [0, 1, nvec // 2 + 1, nvec - 1]
    Xh = np.ascontiguousarray(dX[:, cols].cpu().numpy())
    rng = np.random.default_rng(99 + k)
    rows = _sample_rows(cfg, sysm, rng)
    want = ref.apply_H_rows(Xh, rows)
    got = dY[torch.from_numpy(rows).cuda()][:, cols].cpu().numpy()
    assert np.all(np.isfinite(got))
    assert rel_fro(got, want) < TOL
    # every sampled row on its own (a wrong face / wrap / support row cannot hide in the norm)
    err = np.linalg.norm(got - want, axis=1) / np.maximum(np.linalg.norm(want, axis=1), 1e-300)
    assert float(err.max()) < 1e-10
    del dX, dY, work
    torch.cuda.empty_cache()


@pytest.mark.parametrize("k", [2, 3, 4])
def test_hermiticity_and_product_identity_at_full_size(k):
    """No oracle needed: <x, H y> = conj <y, H x>, and 2 T_j T_k X = T_{j+k} X + T_{|j-k|} X with the bounds the bench uses."""
    import torch
    from paper_2410_02754_b200 import binding
    cfg = synth.CONFIGS[k]
    gpu = binding.Csf(cfg.ncell, cfg.box, cfg.order, cfg.bc, stream=torch.cuda.current_stream().cuda_stream)
    sysm = synth.make_system(cfg, gpu.node_coords(), gpu.mass_diag())
    gpu.set_potential(sysm.veff, sysm.bxyz)
    gpu.set_projectors(sysm.node_ptr, sysm.node_idx, sysm.nproj, sysm.pvals, sysm.atom_type, sysm.delta, sysm.delta_ptr)
    rows_n = 2 * gpu.M; nvec = 32
    work = torch.empty(gpu.workspace_bytes(nvec), dtype=torch.uint8, device="cuda")
    x = _device_block(rows_n, nvec, 7 + k); y = _device_block(rows_n, nvec, 70 + k)
    hx = torch.empty_like(x); hy = torch.empty_like(x)
    gpu.apply_H(x, hx, nvec, nvec, work); gpu.apply_H(y, hy, nvec, nvec, work)
    torch.cuda.synchronize()
    lhs = (x.conj() * hy).sum(0); rhs = (y.conj() * hx).sum(0).conj()
    assert float(((lhs - rhs).abs() / lhs.abs().clamp_min(1e-300)).max()) < 1e-11
    del hx, hy, y

    x1 = torch.empty((rows_n, 1), dtype=torch.complex128, device="cuda"); y1 = torch.empty_like(x1)

    def apply_h_host(v):
        x1.copy_(torch.from_numpy(np.ascontiguousarray(v)).cuda()); gpu.apply_H(x1, y1, 1, 1, work); return y1.cpu().numpy()

    a, b, _, _ = bounds.lanczos_bounds(apply_h_host, rows_n, k=20)
    j, m = 5, 3
    tk = torch.empty_like(x); tjk = torch.empty_like(x); tsum = torch.empty_like(x); tdiff = torch.empty_like(x)
    gpu.filter(x, tk, nvec, nvec, m, a, b, 0, work)
    gpu.filter(tk, tjk, nvec, nvec, j, a, b, 0, work)
    gpu.filter(x, tsum, nvec, nvec, j + m, a, b, 0, work)
    gpu.filter(x, tdiff, nvec, nvec, j - m, a, b, 0, work)
    torch.cuda.synchronize()
    lhs = 2.0 * tjk; rhs = tsum + tdiff
    assert float((lhs - rhs).norm() / rhs.norm()) < 1e-11


ORACLE_COLS = 4      # columns at each end of the block that the oracle filters: {0..3, B-4..B-1}


@pytest.mark.parametrize("k", [2, 3, 4])
def test_filter_at_full_size_against_oracle(k):
    """The launch bench.py times (whole block of the config, ld = nvec = B, the config's degree), both modes, against the
    ORACLE's filter on the columns {0..3, B-4..B-1} (SURVEY 8(d) parity row; eq.70): block Frobenius error
    and per-column maximum. The oracle assembles the global CSR once (17 GB at config 3) and filters the 8 columns copied
    back from the device block, so both sides see bit-identical inputs; a, b are inputs of both sides (Lanczos on apply_H)."""
    import time
    import torch
    from paper_2410_02754_b200 import binding
    cfg = synth.CONFIGS[k]
    t0 = time.perf_counter()
    ref, gpu, sysm = _setup(cfg, sparse=True)
    t_setup = time.perf_counter() - t0
    rows_n = 2 * ref.M; nvec = cfg.nvec
    wb = max(gpu.workspace_bytes(nvec), gpu.workspace_bytes(nvec, binding.CSF_FP32_INTERMEDIATE))
    work = torch.empty(wb, dtype=torch.uint8, device="cuda")
    x1 = torch.empty((rows_n, 1), dtype=torch.complex128, device="cuda"); y1 = torch.empty_like(x1)

    def apply_h_host(v):
        x1.copy_(torch.from_numpy(np.ascontiguousarray(v)).cuda()); gpu.apply_H(x1, y1, 1, 1, work); return y1.cpu().numpy()

    a, b, _, _ = bounds.lanczos_bounds(apply_h_host, rows_n, k=20)
    X = _device_block(rows_n, nvec, 900 + k); Y = torch.empty_like(X)
    cols = list(range(ORACLE_COLS)) + list(range(nvec - ORACLE_COLS, nvec))
    gpu.filter(X, Y, nvec, nvec, cfg.degree, a, b, binding.CSF_FP64, work)
    torch.cuda.synchronize()
    Y64 = Y[:, cols].cpu().numpy()
    gpu.filter(X, Y, nvec, nvec, cfg.degree, a, b, binding.CSF_FP32_INTERMEDIATE, work)
    torch.cuda.synchronize()
    Y32 = Y[:, cols].cpu().numpy()
    Xh = np.ascontiguousarray(X[:, cols].cpu().numpy())
    del X, Y, work, x1, y1
    torch.cuda.empty_cache()
    t0 = time.perf_counter()
    Yref = ref.filter(Xh, cfg.degree, a, b)
    t_ref = time.perf_counter() - t0
    e64, c64 = assert_block_close(Y64, Yref, TOL, col_tol=1e-10)
    e32, c32 = assert_block_close(Y32, Yref, 1e-5, col_tol=1e-4)
    assert e32 > 1e-9          # it really is the single-precision path
    print(f"config {k}: FP64 rel Frobenius {e64:.2e} (column max {c64:.2e}); FP32-intermediate {e32:.2e} (column max {c32:.2e}); "
          f"oracle set-up {t_setup:.0f} s, oracle filter of {len(cols)} columns {t_ref:.0f} s")

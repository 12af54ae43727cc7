"""csf_apply_H_static, the allocation-free entry point (include/csf.h): its output against csf_apply_H's on the same
inputs, on two calls in a row (the static scratch keeps the first call's contents), and its size limit.

Collected last on purpose (pytest -x: a failure here must not hide the parity tests).
Tolerance: the relative Frobenius error <= 1e-11 of the other FP64 parity tests (test_gpu_parity.py); the two paths run
the same kernels, the only difference between them is the order of the scatter-add."""
import numpy as np
import pytest

from paper_2410_02754_b200 import synth, binding
from helpers import setup_pair, gpu_apply_H, assert_block_close

pytestmark = pytest.mark.gpu
TOL = 1e-11


def _static_apply(gpu, X, ld=None):
    import torch
    nvec = X.shape[1]; ld = ld or nvec
    dX = torch.zeros((X.shape[0], ld), dtype=torch.complex128, device="cuda"); dX[:, :nvec] = torch.from_numpy(X).cuda()
    dY = torch.full((X.shape[0], ld), 7.0 + 3.0j, dtype=torch.complex128, device="cuda")
    gpu.apply_H_static(dX, dY, ld, nvec)
    torch.cuda.synchronize()
    out = dY.cpu().numpy()
    if ld > nvec:
        assert np.all(out[:, nvec:] == 7.0 + 3.0j), "padding columns were touched"
    return out[:, :nvec].copy()


CASES = [synth.CONFIGS[0],
         synth.Config(9, "p4_dirichlet_z", (4, 3, 5), (8.0, 6.0, 10.0), 4, (0, 0, 1), 3, "uniform", 13, 6, 0, 4242)]


@pytest.mark.parametrize("cfg", CASES, ids=lambda c: c.name)
def test_static_entry_matches_workspace_path_twice(cfg):
    ref, gpu, s = setup_pair(cfg)
    M2 = 2 * ref.M
    # first call: the full block; second call, straight after: other data, fewer vectors, padded rows
    # (the scratch still holds the first call's coefficients where the second does not reach)
    X1 = synth.random_block(s.rng, M2, cfg.nvec)
    X2 = synth.random_block(s.rng, M2, 5)
    Y1 = _static_apply(gpu, X1)
    Y2 = _static_apply(gpu, X2, ld=8)
    assert_block_close(Y1, gpu_apply_H(gpu, X1), TOL)
    assert_block_close(Y2, gpu_apply_H(gpu, X2, ld=8), TOL)
    assert_block_close(Y1, ref.apply_H(X1), TOL)
    assert_block_close(Y2, ref.apply_H(X2), TOL)
    # and once more with the first block: same answer as before the scratch was reused
    assert_block_close(_static_apply(gpu, X1), Y1, TOL)


def test_static_entry_allocates_nothing():
    """Free device memory is the same before and after a repeated call (the first call of a shape may load kernels)."""
    import torch
    cfg = CASES[0]
    ref, gpu, s = setup_pair(cfg)
    X = torch.from_numpy(synth.random_block(s.rng, 2 * ref.M, cfg.nvec)).cuda()
    Y = torch.empty_like(X)
    gpu.apply_H_static(X, Y, cfg.nvec, cfg.nvec)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        gpu.apply_H_static(X, Y, cfg.nvec, cfg.nvec)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0


def test_static_entry_rejects_sizes_beyond_its_scratch():
    import torch
    cfg = CASES[0]
    ref, gpu, s = setup_pair(cfg)
    nvec = 6000                      # 2 atoms x 18 projectors: C and C~ need about 1.9 kB per vector, the limit is 8 MiB
    X = torch.zeros((2 * ref.M, nvec), dtype=torch.complex128, device="cuda")
    Y = torch.zeros_like(X)
    with pytest.raises(binding.CsfError) as ei:
        gpu.apply_H_static(X, Y, nvec, nvec)
    assert ei.value.code == binding.CSF_EUNSUPPORTED
    msg = str(ei.value)
    assert "static limit" in msg and str(binding.STATIC_SCRATCH_BYTES) in msg and "6000" in msg
    torch.cuda.synchronize()
    assert float(Y.abs().max()) == 0.0                      # nothing was launched
    # the same context still serves a size that fits
    Xs = synth.random_block(s.rng, 2 * ref.M, 7)
    assert_block_close(_static_apply(gpu, Xs), gpu_apply_H(gpu, Xs), TOL)
    # without projectors there is no scratch and no limit from it
    gpu.set_projectors([0], [], [], [], [], [], [0]); ref.set_projectors([0], [], [], [], [], [], [0])
    assert_block_close(_static_apply(gpu, Xs), ref.apply_H(Xs), TOL)

"""Every column-kernel variant against the oracle: the cell-per-iteration kernel with 4 vectors per CTA (16 lanes) and with 8
(32 lanes, orders 4 and 5), the warp-specialised streaming kernel (csf_colws.cuh, orders 4 and 5, 32 lanes) and the fused
half-block path of csf_filter (order 5: column kernel with gather warps; CSF_FUSED_GATHER=1 forces it at small sizes). By default
libcsf picks the variant; CSF_LANES / CSF_KERNEL pin it at csf_create, so every case below runs
through each kernel."""
import numpy as np
import pytest

from paper_2410_02754_b200 import bounds, synth
from helpers import gpu_apply_H, gpu_filter, rel_fro, setup_pair, assert_block_close
from test_gpu_parity import TOL, TOL32, _cfg, gpu_filter32

pytestmark = pytest.mark.gpu


@pytest.fixture(params=[16, 32, "ws", "fused"])
def lanes(request, monkeypatch):
    """16: 4 vectors per CTA; 32: 8 vectors per CTA (cell-per-iteration kernel); "ws": the warp-specialised streaming kernel;
    "fused": csf_filter's half-block path (order 5, complex128: the column kernel with two gather warps that compute the
    projector coefficients of the other half-block) forced for every block size, which the policy takes for blocks that are multiples of 64 vectors."""
    if request.param == "ws":
        monkeypatch.setenv("CSF_KERNEL", "ws")
    elif request.param == "fused":
        monkeypatch.setenv("CSF_LANES", "32")
        monkeypatch.setenv("CSF_FUSED_GATHER", "1")
    else:
        monkeypatch.setenv("CSF_LANES", str(request.param))
    return request.param


@pytest.mark.parametrize("order", [4, 5])
@pytest.mark.parametrize("bc", [(0, 0, 0), (0, 0, 1), (1, 0, 0)])
@pytest.mark.parametrize("nvec,ld", [(5, 9), (8, 8), (16, 16), (19, 24)])
def test_apply_H_pinned_lanes(lanes, order, bc, nvec, ld):
    """Ragged and full vector chunks (8 | nvec or not), periodic / Dirichlet faces, non-cubic cells."""
    cfg = _cfg((2, 3, 2), (2.2, 3.0, 1.9), order, bc, 2, nvec=nvec)
    ref, gpu, s = setup_pair(cfg)
    X = synth.random_block(s.rng, 2 * ref.M, nvec)
    assert_block_close(gpu_apply_H(gpu, X, ld=ld), ref.apply_H(X), TOL)


@pytest.mark.parametrize("seg_len,chunk_group", [(0, 16), (1, 1), (2, 2), (3, 1), (3, 2)])
@pytest.mark.parametrize("base,ncell,natoms,nvec,degree", [(2, (4, 4, 8), 3, 24, 10), (3, (6, 6, 6), 4, 16, 12), (4, (6, 6, 6), 4, 16, 12)])
def test_filter_pinned_lanes_shapes_of_large_configs(lanes, base, ncell, natoms, nvec, degree, seg_len, chunk_group):
    """Sub-meshes of configs 2-4 (Dirichlet z and non-cubic cells included) through both kernels and both modes, with the
    traversal hooks set so that what only full-size meshes reach by default runs here: several z-segments per column
    (seg_len 1, 2, 3 on 6 or 8 cells: the z-face handed over through global memory, the final-carry flush, a ragged last
    segment) and several chunk groups (chunk_group 1, 2 with 2-6 vector chunks)."""
    cfg = synth.scaled_config(synth.CONFIGS[base], ncell, natoms, nvec=nvec, degree=degree)
    ref, gpu, s = setup_pair(cfg)
    gpu.set_tuning(seg_len, chunk_group)
    a, b, _, _ = bounds.lanczos_bounds(lambda v: ref.apply_H(v), 2 * ref.M)
    X = synth.random_block(s.rng, 2 * ref.M, nvec)
    Yref = ref.filter(X, degree, a, b)
    assert_block_close(gpu_filter(gpu, X, degree, a, b), Yref, TOL)
    assert_block_close(gpu_filter32(gpu, X, degree, a, b), Yref, TOL32)
    assert_block_close(gpu_filter(gpu, X[:, :nvec - 3], degree, a, b, ld=nvec), Yref[:, :nvec - 3], TOL)      # ragged last chunk


@pytest.mark.parametrize("seg_len", [1, 2, 5])
@pytest.mark.parametrize("bc", [(0, 0, 0), (0, 0, 1), (1, 1, 0)])
def test_apply_H_segment_boundaries(lanes, bc, seg_len):
    """One H apply with the z-face of every segment boundary checked row by row (not only in the block norm)."""
    cfg = _cfg((2, 2, 5), (2.0, 2.4, 4.5), 5, bc, 2, nvec=9)
    ref, gpu, s = setup_pair(cfg)
    gpu.set_tuning(seg_len, 1)
    X = synth.random_block(s.rng, 2 * ref.M, 9)
    Y = gpu_apply_H(gpu, X, ld=12); Yref = ref.apply_H(X)
    assert_block_close(Y, Yref, TOL)
    err = np.linalg.norm(Y - Yref, axis=1) / np.maximum(np.linalg.norm(Yref, axis=1), 1e-300)
    assert float(err.max()) < 1e-10


def test_run_to_run_spread_is_reported(lanes):
    """The assembly adds shared-face contributions with RED.F64, whose order is not fixed: results are NOT bitwise repeatable
    (DESIGN.md section 4). The spread between two runs is reported and bounded far below the parity tolerance."""
    cfg = synth.scaled_config(synth.CONFIGS[3], (6, 6, 6), 4, nvec=16, degree=12)
    ref, gpu, s = setup_pair(cfg)
    a, b, _, _ = bounds.lanczos_bounds(lambda v: ref.apply_H(v), 2 * ref.M)
    X = synth.random_block(s.rng, 2 * ref.M, 16)
    Y1 = gpu_filter(gpu, X, 12, a, b); Y2 = gpu_filter(gpu, X, 12, a, b)
    spread = rel_fro(Y1, Y2)
    print(f"run-to-run spread (lanes {lanes}): relative Frobenius {spread:.3e}, bitwise equal: {np.array_equal(Y1, Y2)}")
    assert spread < 1e-13


def test_policy_and_pinned_variants_agree():
    """The variant libcsf picks on its own gives the oracle's result too (FP64 and FP32-intermediate on one context)."""
    cfg = synth.scaled_config(synth.CONFIGS[2], (4, 4, 8), 3, nvec=24, degree=6)
    ref, gpu, s = setup_pair(cfg)
    a, b, _, _ = bounds.lanczos_bounds(lambda v: ref.apply_H(v), 2 * ref.M)
    X = synth.random_block(s.rng, 2 * ref.M, 24)
    Yref = ref.filter(X, 6, a, b)
    assert_block_close(gpu_filter(gpu, X, 6, a, b), Yref, TOL)
    assert_block_close(gpu_filter32(gpu, X, 6, a, b), Yref, TOL32)
    assert_block_close(gpu_filter(gpu, X[:, :13], 6, a, b, ld=16), Yref[:, :13], TOL)


def test_column_lanes_query(monkeypatch):
    """csf_column_lanes reports the variant a call runs with: the measured policy by default, CSF_LANES pins it."""
    from paper_2410_02754_b200 import binding
    monkeypatch.delenv("CSF_LANES", raising=False)
    slab = binding.Csf((2, 2, 3), (4.0, 4.0, 6.0), 5, (0, 0, 1))
    bulk = binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 5, (0, 0, 0))
    p4 = binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 4, (0, 0, 0))
    p3 = binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 3, (0, 0, 0))
    for ctx in (slab, bulk, p4):
        for mode in (binding.CSF_FP64, binding.CSF_FP32_INTERMEDIATE):
            assert ctx.column_lanes(16, mode) == 32 and ctx.column_lanes(13, mode) == 32
    assert p3.column_lanes(16, binding.CSF_FP64) == 16
    monkeypatch.setenv("CSF_LANES", "16")
    assert binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 5, (0, 0, 0)).column_lanes(16, binding.CSF_FP64) == 16
    monkeypatch.setenv("CSF_LANES", "32")
    assert binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 5, (0, 0, 0)).column_lanes(16, binding.CSF_FP32_INTERMEDIATE) == 32
    assert binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 3, (0, 0, 0)).column_lanes(16, binding.CSF_FP64) == 16
    monkeypatch.delenv("CSF_LANES")
    monkeypatch.setenv("CSF_KERNEL", "ws")
    assert binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 4, (0, 0, 0)).column_lanes(16, binding.CSF_FP64) == 32


def test_fused_gather_policy_and_agreement(monkeypatch):
    """csf_filter_fused_gather reports the path a block takes (policy: complex128, order 5, 18 projectors per atom, a multiple
    of 64 vectors; CSF_FUSED_GATHER pins it), and the fused and the unfused path give the oracle's result on the same blocks:
    64 vectors (the policy's own choice, halves 32 + 32) and 67 (forced, split 40 + 27 with a ragged second half)."""
    from paper_2410_02754_b200 import binding
    for v in ("CSF_LANES", "CSF_KERNEL", "CSF_FUSED_GATHER"):
        monkeypatch.delenv(v, raising=False)
    cfg = synth.scaled_config(synth.CONFIGS[3], (4, 4, 4), 2, nvec=67, degree=7)
    ref, gpu, s = setup_pair(cfg)
    assert gpu.filter_fused_gather(64, binding.CSF_FP64) and gpu.filter_fused_gather(256, binding.CSF_FP64)
    assert not gpu.filter_fused_gather(63, binding.CSF_FP64) and not gpu.filter_fused_gather(96, binding.CSF_FP64)
    assert not gpu.filter_fused_gather(64, binding.CSF_FP32_INTERMEDIATE)
    a, b, _, _ = bounds.lanczos_bounds(lambda v: ref.apply_H(v), 2 * ref.M)
    X = synth.random_block(s.rng, 2 * ref.M, 67)
    Yref = ref.filter(X, 7, a, b)
    Yp = gpu_filter(gpu, X[:, :64], 7, a, b, ld=70)                     # the policy's fused path
    assert_block_close(Yp, Yref[:, :64], TOL)
    monkeypatch.setenv("CSF_FUSED_GATHER", "0")
    ref2, gpu2, _ = setup_pair(cfg)
    assert not gpu2.filter_fused_gather(64, binding.CSF_FP64)
    Yu = gpu_filter(gpu2, X, 7, a, b, ld=70)
    assert_block_close(Yu, Yref, TOL)
    assert rel_fro(Yp, Yu[:, :64]) < 1e-13
    monkeypatch.setenv("CSF_FUSED_GATHER", "1")
    p4 = binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 4, (0, 0, 0))
    assert not p4.filter_fused_gather(256, binding.CSF_FP64)          # order 4 has no kernel with gather warps
    # forced on, the path starts at 9 vectors (halves of 8 + 1: the first half must be a multiple of 8 vectors)
    ref3, gpu3, _ = setup_pair(cfg)
    assert gpu3.filter_fused_gather(9, binding.CSF_FP64) and not gpu3.filter_fused_gather(8, binding.CSF_FP64)
    for n in (8, 9, 10):
        assert_block_close(gpu_filter(gpu3, X[:, :n], 7, a, b, ld=12), Yref[:, :n], TOL)
    Yf = gpu_filter(gpu3, X, 7, a, b, ld=70)                             # 67 = 40 + 27
    assert_block_close(Yf, Yref, TOL)
    assert rel_fro(Yf, Yu) < 1e-13


@pytest.mark.parametrize("gather", ["reg", "bulk"])
@pytest.mark.parametrize("base,ncell,natoms,nvec,degree", [(2, (4, 4, 8), 3, 24, 6), (4, (6, 6, 6), 4, 13, 8)])
def test_both_projector_gather_kernels(monkeypatch, gather, base, ncell, natoms, nvec, degree):
    """The projector gather (a5) has two kernels: src rows staged in shared memory by bulk copies (the default for complex128
    and complex64 blocks alike) and plain register loads (CSF_GATHER=reg pins it). Both against the oracle, both precision
    modes, full and ragged blocks (13 vectors: the complex64 rows are copied up to the even pad column)."""
    monkeypatch.setenv("CSF_GATHER", gather)
    cfg = synth.scaled_config(synth.CONFIGS[base], ncell, natoms, nvec=nvec, degree=degree)
    ref, gpu, s = setup_pair(cfg)
    a, b, _, _ = bounds.lanczos_bounds(lambda v: ref.apply_H(v), 2 * ref.M)
    X = synth.random_block(s.rng, 2 * ref.M, nvec)
    Yref = ref.filter(X, degree, a, b)
    assert_block_close(gpu_filter(gpu, X, degree, a, b), Yref, TOL)
    assert_block_close(gpu_filter32(gpu, X, degree, a, b), Yref, TOL32)
    assert_block_close(gpu_apply_H(gpu, X, ld=nvec + 3), ref.apply_H(X), TOL)


def test_filter_host_with_fused_chunks(monkeypatch):
    """csf_filter_host on an order-5 mesh with a block wide enough for its 64-column chunks to take the fused half-block path by
    the policy itself (200 columns: chunks of 32, 64, 64, 8, 32; the half chunks at both ends and the remainder run unfused)."""
    import torch
    for v in ("CSF_LANES", "CSF_KERNEL", "CSF_FUSED_GATHER"):
        monkeypatch.delenv(v, raising=False)
    cfg = synth.scaled_config(synth.CONFIGS[3], (4, 4, 4), 2, nvec=200, degree=5)
    ref, gpu, s = setup_pair(cfg)
    a, b, _, _ = bounds.lanczos_bounds(lambda v: ref.apply_H(v), 2 * ref.M)
    X = synth.random_block(s.rng, 2 * ref.M, 200)
    hX = torch.zeros((2 * ref.M, 204), dtype=torch.complex128).pin_memory(); hX[:, :200] = torch.from_numpy(X)
    hY = torch.full((2 * ref.M, 204), 7.0 + 3.0j, dtype=torch.complex128).pin_memory()
    gpu.set_host_chunk(64)
    gpu.filter_host(hX, hY, 204, 200, 5, a, b)
    out = hY.numpy()
    assert_block_close(out[:, :200], ref.filter(X, 5, a, b), TOL)
    assert np.all(out[:, 200:] == 7.0 + 3.0j), "padding columns were touched"

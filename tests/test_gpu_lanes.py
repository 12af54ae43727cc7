"""Both column-kernel variants — 4 vectors per CTA (16 lanes) and 8 vectors per CTA (32 lanes, orders 4 and 5) — against
the oracle. By default libcsf picks the variant per call; CSF_LANES pins it at csf_create, so every
case below runs through each kernel whatever the policy is."""
import numpy as np
import pytest

from paper_2410_02754_b200 import bounds, synth
from helpers import gpu_apply_H, gpu_filter, rel_fro, setup_pair
from test_gpu_parity import TOL, TOL32, _cfg, gpu_filter32

pytestmark = pytest.mark.gpu


@pytest.fixture(params=[16, 32])
def lanes(request, monkeypatch):
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
    assert rel_fro(gpu_apply_H(gpu, X, ld=ld), ref.apply_H(X)) < TOL


@pytest.mark.parametrize("base,ncell,natoms,nvec,degree", [(2, (4, 4, 8), 3, 24, 10), (3, (6, 6, 6), 4, 16, 12), (4, (6, 6, 6), 4, 16, 12)])
def test_filter_pinned_lanes_shapes_of_large_configs(lanes, base, ncell, natoms, nvec, degree):
    cfg = synth.scaled_config(synth.CONFIGS[base], ncell, natoms, nvec=nvec, degree=degree)
    ref, gpu, s = setup_pair(cfg)
    a, b, _, _ = bounds.lanczos_bounds(lambda v: ref.apply_H(v), 2 * ref.M)
    X = synth.random_block(s.rng, 2 * ref.M, nvec)
    Yref = ref.filter(X, degree, a, b)
    assert rel_fro(gpu_filter(gpu, X, degree, a, b), Yref) < TOL
    assert rel_fro(gpu_filter32(gpu, X, degree, a, b), Yref) < TOL32


def test_policy_and_pinned_variants_agree():
    """The variant libcsf picks on its own gives the oracle's result too (FP64 and FP32-intermediate on one context)."""
    cfg = synth.scaled_config(synth.CONFIGS[2], (4, 4, 8), 3, nvec=24, degree=6)
    ref, gpu, s = setup_pair(cfg)
    a, b, _, _ = bounds.lanczos_bounds(lambda v: ref.apply_H(v), 2 * ref.M)
    X = synth.random_block(s.rng, 2 * ref.M, 24)
    Yref = ref.filter(X, 6, a, b)
    assert rel_fro(gpu_filter(gpu, X, 6, a, b), Yref) < TOL
    assert rel_fro(gpu_filter32(gpu, X, 6, a, b), Yref) < TOL32
    assert rel_fro(gpu_filter(gpu, X[:, :13], 6, a, b, ld=16), Yref[:, :13]) < TOL


def test_column_lanes_query(monkeypatch):
    """csf_column_lanes reports the variant a call runs with: the measured policy by default, CSF_LANES pins it."""
    from paper_2410_02754_b200 import binding
    monkeypatch.delenv("CSF_LANES", raising=False)
    slab = binding.Csf((2, 2, 3), (4.0, 4.0, 6.0), 5, (0, 0, 1))
    bulk = binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 5, (0, 0, 0))
    p4 = binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 4, (0, 0, 0))
    p3 = binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 3, (0, 0, 0))
    assert slab.column_lanes(16, binding.CSF_FP64) == 32 and slab.column_lanes(16, binding.CSF_FP32_INTERMEDIATE) == 32
    assert bulk.column_lanes(16, binding.CSF_FP64) == 32 and bulk.column_lanes(16, binding.CSF_FP32_INTERMEDIATE) == 16
    assert bulk.column_lanes(13, binding.CSF_FP32_INTERMEDIATE) == 32          # ragged block: general mode
    assert p4.column_lanes(16, binding.CSF_FP64) == 32 and p4.column_lanes(16, binding.CSF_FP32_INTERMEDIATE) == 32
    assert p3.column_lanes(16, binding.CSF_FP64) == 16
    monkeypatch.setenv("CSF_LANES", "16")
    assert binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 5, (0, 0, 0)).column_lanes(16, binding.CSF_FP64) == 16
    monkeypatch.setenv("CSF_LANES", "32")
    assert binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 5, (0, 0, 0)).column_lanes(16, binding.CSF_FP32_INTERMEDIATE) == 32
    assert binding.Csf((2, 2, 2), (4.0, 4.0, 4.0), 3, (0, 0, 0)).column_lanes(16, binding.CSF_FP64) == 16

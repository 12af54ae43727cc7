import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def cfg0_oracle():
    """Config 0 (BASELINE.json configs[0]) set up on the oracle: ctx, synthetic system, bounds."""
    from oracle import oracle as O
    from paper_2410_02754_b200 import synth, bounds
    cfg = synth.CONFIGS[0]
    ctx = O.RefCtx(cfg.ncell, cfg.box, cfg.order, cfg.bc)
    sys_ = synth.make_system(cfg, ctx.node_coords(), ctx.mass_diag())
    ctx.set_potential(sys_.veff, sys_.bxyz)
    ctx.set_projectors(sys_.node_ptr, sys_.node_idx, sys_.nproj, sys_.pvals, sys_.atom_type, sys_.delta, sys_.delta_ptr)
    a, b, _, _ = bounds.lanczos_bounds(lambda v: ctx.apply_H(v), 2 * ctx.M)
    X = synth.random_block(sys_.rng, 2 * ctx.M, cfg.nvec)
    return dict(cfg=cfg, ctx=ctx, sys=sys_, a=a, b=b, X=X)

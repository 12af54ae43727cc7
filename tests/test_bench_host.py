"""Host logic of bench.py: state sharding over ranks (replicas, no data-path collective), the flop model, the
bounded CPU sample, and the max-over-ranks timing reduction under a world_size-2 gloo group on CPU."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402
from paper_2410_02754_b200 import synth  # noqa: E402


def test_shard_states_partitions_all_blocks():
    for nstates, nvec, world in [(7700, 256, 1), (7700, 256, 2), (22000, 256, 8), (16, 16, 4), (5500, 512, 3)]:
        seen = []
        for r in range(world):
            seen += bench.shard_states(nstates, nvec, r, world)
        nblocks = -(-nstates // nvec)
        assert sorted(seen) == list(range(nblocks))          # every block exactly once, no overlap
    assert bench.shard_states(7700, 256, 1, 2)[0] == 1


def test_flop_model_matches_survey_table():
    # rank-one variant (12 n^4 + 40 n^3) / p^3, + 144 c_ov + 24
    cell, gather, total = bench.algorithmic_flops(5, 1.0)
    assert abs((12 * 6 ** 4 + 40 * 6 ** 3) / 125 - 193.54) < 0.01
    assert abs(total - (193.536 + 144 + 24)) < 1e-9 and abs(gather - 72) < 1e-12 and abs(cell + gather - total) < 1e-12
    assert abs(bench.algorithmic_flops(4, 0.0)[2] - ((12 * 625 + 40 * 125) / 64 + 24)) < 1e-9


def test_cpu_sample_keeps_cell_size_order_bc_and_density():
    for k in (2, 3, 4):
        cfg = synth.CONFIGS[k]; sc = bench.cpu_sample_config(cfg)
        assert sc.order == cfg.order and sc.bc == cfg.bc and sc.degree == cfg.degree
        for d in range(3):
            assert abs(sc.box[d] / sc.ncell[d] - cfg.box[d] / cfg.ncell[d]) < 1e-12
        dens = cfg.natoms / (cfg.ncell[0] * cfg.ncell[1] * cfg.ncell[2])
        assert abs(sc.natoms - dens * sc.ncell[0] * sc.ncell[1] * sc.ncell[2]) <= 1.0
    assert bench.cpu_sample_config(synth.CONFIGS[0]).ncell == synth.CONFIGS[0].ncell


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    blocks = bench.shard_states(7700, 256, rank, world)
    local_ms = 10.0 + 5.0 * rank                          # rank 1 is the slow one
    ms = bench.reduce_max_time(local_ms, dist)
    out.put((rank, blocks, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_timing_and_sharding():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, b0, ms0), (r1, b1, ms1) = res
    assert ms0 == ms1 == 15.0                               # max over ranks on both
    assert set(b0).isdisjoint(b1) and sorted(b0 + b1) == list(range(31))
    assert len(b0) == 16 and len(b1) == 15


def test_reference_arm_runs_only_on_rank0(monkeypatch, capsys):
    import argparse
    monkeypatch.setenv("RANK", "1")
    args = argparse.Namespace(config=0, steps=1, warmup=0, gpus=2)
    assert bench.main_reference(args) == 0
    assert capsys.readouterr().out == ""

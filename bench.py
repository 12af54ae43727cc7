#!/usr/bin/env python
"""bench.py — throughput of the Chebyshev-filtered spinor H.X (csf_filter) on B200, one JSON line.

A "step" is one pass of the whole hot path over one block: Y = T_m(H~) X for B spinor vectors, i.e. m
applications of [projector gather -> Delta -> gather/cell apply/assembly/recurrence].
metric = spinor DoF x vectors x degree per second (BASELINE.json). Headline workload: BASELINE.json configs[3]
(periodic bulk, 32^3 cells of order 5, 8.19 M spinor DoF, 500 atoms, block of 256, degree 40), the largest
single-GPU configuration of the roofline target set; `--config k` selects another. The same JSON line carries the other
roofline-target legs (`other_configs`: configs 2 and 4 in complex128, config 4 FP32-intermediate), the Rayleigh-Ritz /
density timings on the filtered block (`subspace`), the end-to-end leg through host buffers (`e2e`) and the CPU oracle
on the config's own operator (`cpu_baseline`). DESIGN.md section 6 describes every field.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--mode fp64|fp32] [--impl ours|reference]

N > 1 (under torchrun): the path does not shard (BASELINE.json north_star), so every rank filters its own block
of states on its own replica of the operator ("replicas only"; the paper's band groups). No
data-path collective; the only communication is the timing barrier / max-over-ranks.

--impl reference times the CPU oracle (oracle/) on the host cores on a bounded sample of the same workload.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2410_02754_b200 import synth  # noqa: E402

METRIC = "Cheb-filtered spinor HX: DoF*vectors*degree/s"
UNIT = "DoF*vec*deg/s"
FP64_FMA_PER_CLK_PER_SM = 64          # 4 SMSPs x 16 FP64 lanes (B200 data sheet: 37-40 TF/s FP64 vector at 1.97 GHz)
SM_COUNT = 148


# ----------------------------------------------------------------------------------------------- helpers
def algorithmic_flops(p, c_ov):
    """FP64 flops per unit (one spinor DoF x vector x degree) of the algorithm the kernels implement (DESIGN.md
    'Roofline'): sum-factorised 1/2 K with the rank-one mass form, nodal 2x2 potential, projector gather + expand,
    recurrence. Returns (cell kernel, projector gather kernel, total)."""
    n = p + 1
    kin = (12.0 * n ** 4 + 40.0 * n ** 3) / p ** 3      # 3 dense + 4 rank-one 1-D contractions, re and im
    pot, rec = 14.0, 10.0
    expand = 72.0 * c_ov                                # 18 projectors x 2 flops x (re, im) per support row per spin-vector
    gather = 72.0 * c_ov
    return kin + pot + rec + expand, gather, kin + pot + rec + expand + gather


def shard_states(nstates, nvec, rank, world):
    """Block indices (of ceil(nstates / nvec) blocks of `nvec` states) owned by `rank`: round robin, no exchange."""
    nblocks = max(1, math.ceil(nstates / nvec))
    return [b for b in range(nblocks) if b % world == rank]


def reduce_max_time(ms, dist_mod=None):
    """Max over ranks of a local duration (the only cross-rank operation of the benchmark)."""
    if dist_mod is None or not dist_mod.is_initialized():
        return ms
    import torch
    dev = "cuda" if dist_mod.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms], dtype=torch.float64, device=dev)
    dist_mod.all_reduce(t, op=dist_mod.ReduceOp.MAX)
    return float(t.item())


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons every 200 ms while the timed region runs."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, device):
        self.device, self.proc, self.lines = device, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200", "-i", str(self.device)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True); self.thr.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)), "samples": len(sm), "reasons": sorted(reasons)}


def build_system(cfg, ctx, with_projectors=True):
    """Seeded synthetic operator inputs for `cfg` on node coordinates / masses exported by `ctx` (either side)."""
    sysm = synth.make_system(cfg, ctx.node_coords(), ctx.mass_diag(), with_projectors=with_projectors)
    ctx.set_potential(sysm.veff, sysm.bxyz)
    if with_projectors:
        ctx.set_projectors(sysm.node_ptr, sysm.node_idx, sysm.nproj, sysm.pvals, sysm.atom_type, sysm.delta, sysm.delta_ptr)
    return sysm


def roofline_model(p, c_ov, fp32):
    """Algorithmic bytes and flops per unit and the time floors they imply.
    FP64 mode: 48 B/unit through the column kernel + 16 c_ov B/unit re-read by the projector gather; all flops FP64.
    FP32-intermediate mode: 24 B/unit + 8 c_ov; the cell arithmetic (kinetic, potential, recurrence) runs on the FP32 FMA pipe,
    the projector contractions (gather + expansion, 144 c_ov flops/unit) stay FP64."""
    f_cell, f_gather, f_total = algorithmic_flops(p, c_ov)
    f_proj = 144.0 * c_ov
    return {"bytes_column": 24.0 if fp32 else 48.0, "bytes_gather": (8.0 if fp32 else 16.0) * c_ov,
            "flops_fp64": f_proj if fp32 else f_total, "flops_fp32": (f_total - f_proj) if fp32 else 0.0,
            "flops_column": f_cell, "flops_total": f_total}


def cpu_sample_config(cfg):
    """Fallback sample when the host cannot hold the config's CSR: same cell size, order, boundary conditions, atom density
    and degree on an 8x8x8-cell sub-mesh (config 0/1: the whole mesh), 16 columns."""
    if cfg.index <= 1:
        return synth.Config(cfg.index, cfg.name, cfg.ncell, cfg.box, cfg.order, cfg.bc, cfg.natoms, cfg.placement, min(cfg.nvec, 16), cfg.degree, 0, cfg.seed)
    nc = tuple(min(8, c) for c in cfg.ncell)
    frac = float(np.prod(nc)) / float(np.prod(cfg.ncell))
    return synth.scaled_config(cfg, nc, max(1, int(round(cfg.natoms * frac))), nvec=16, degree=cfg.degree)


class OracleSample:
    """The oracle as it stands (oracle/, OpenMP on all host cores) on a bounded sample of the benchmarked workload:
    the ACTUAL config (mesh, atoms, potential: the global CSR is assembled once, outside the timed region, like the GPU
    side's set-up) with 8 columns and as many Chebyshev degrees as fit `budget_s` seconds (SURVEY 8(d) "CPU baseline").
    If the host cannot hold the CSR it falls back to an 8x8x8-cell sub-mesh and says so."""

    def __init__(self, cfg, budget_s=20.0, est_units_per_s=4.5e7):
        import psutil
        from oracle import oracle as O
        from paper_2410_02754_b200 import bounds
        self.O = O
        need = cfg.M * ((cfg.order + 2) ** 3 * 12.0 + 200.0) + 5 * 2 * cfg.M * 8 * 16.0          # CSR + conn + vectors
        self.full = psutil.virtual_memory().available > 1.5 * need
        self.cfg = cfg
        sc = cfg if self.full else cpu_sample_config(cfg)
        self.ncols = 8 if self.full else sc.nvec
        per_degree = 2.0 * sc.M * self.ncols
        self.degree = int(min(sc.degree, max(2, round(budget_s * est_units_per_s / per_degree)))) if self.full else sc.degree
        self.ref = O.RefCtx(sc.ncell, sc.box, sc.order, sc.bc)
        self.sysm = build_system(sc, self.ref)
        self.a, self.b, _, _ = bounds.lanczos_bounds(lambda v: self.ref.apply_H(v), 2 * self.ref.M, k=6)
        self.X = synth.random_block(self.sysm.rng, 2 * self.ref.M, self.ncols)
        self.units = 2.0 * self.ref.M * self.ncols * self.degree
        if self.full:
            self.desc = (f"the config's own operator ({sc.ncell[0]}x{sc.ncell[1]}x{sc.ncell[2]} cells, {sc.natoms} atoms; CSR assembled outside the timed region), "
                         f"8 columns, degree {self.degree} of {cfg.degree}: {self.units:.3g} of the block's {2.0 * cfg.M * cfg.nvec * cfg.degree:.3g} units; "
                         f"a full block would take {cfg.nvec / 8.0 * cfg.degree / self.degree:.0f}x as long (linear extrapolation)")
        else:
            self.desc = (f"host memory too small for the config's CSR: {sc.ncell[0]}x{sc.ncell[1]}x{sc.ncell[2]} cells of order {sc.order} (same cell size, bc, atom density: "
                         f"{sc.natoms} atoms), {sc.nvec} columns, degree {sc.degree}: {self.units:.3g} of the workload's {2.0 * cfg.M * cfg.nvec * cfg.degree:.3g} units")

    def step(self):
        t0 = time.perf_counter()
        self.ref.filter(self.X, self.degree, self.a, self.b)
        return time.perf_counter() - t0


def run_oracle_sample(cfg, steps=1, warmup=0, budget_s=20.0):
    """Returns (units/s, description, cores, ms/step)."""
    smp = OracleSample(cfg, budget_s=budget_s)
    for _ in range(warmup):
        smp.ref.filter(smp.X[:, :2], 1, smp.a, smp.b)
    dt = sum(smp.step() for _ in range(steps)) / steps
    return smp.units / dt, smp.desc, smp.O.num_threads(), dt * 1e3


def workload_dict(cfg, sysm=None):
    d = {"workload": f"BASELINE.json configs[{cfg.index}] {cfg.name}", "ncell": list(cfg.ncell), "order": cfg.order,
         "bc": ["periodic" if b == 0 else "dirichlet" for b in cfg.bc], "spinor_dof": 2 * cfg.M, "block_vectors": cfg.nvec,
         "degree": cfg.degree, "atoms": cfg.natoms, "projectors_per_atom": synth.N_PROJ,
         "l2": "inputs larger than L2 (block buffers of %.2f GB each)" % (2 * cfg.M * cfg.nvec * 16 / 1e9)}
    if sysm is not None:
        d["c_ov"] = round(sysm.coverage, 4)
    return d


# ----------------------------------------------------------------------------------------------- reference arm
def main_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = synth.CONFIGS[args.config]
    nsteps = max(1, args.steps)
    val, desc, cores, ms = run_oracle_sample(cfg, steps=nsteps, warmup=min(args.warmup, 1), budget_s=max(2.0, min(20.0, 150.0 / (nsteps + 1))))
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": workload_dict(cfg),
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(out))
    return 0


# ----------------------------------------------------------------------------------------------- our arm
def measure(cfg_index, mode_name, steps, warmup, args, ctxs):
    """One benchmark leg: `steps` timed csf_filter calls of one block of config `cfg_index` in `mode_name` on this rank's GPU.
    Returns the result dict and the live objects the end-to-end leg reuses (ctx, X, bounds)."""
    import torch
    import torch.distributed as dist
    from paper_2410_02754_b200 import binding, bounds
    world, rank, local = ctxs["world"], ctxs["rank"], ctxs["local"]
    cfg = synth.CONFIGS[cfg_index]
    nvec = args.nvec or cfg.nvec
    degree = args.degree or cfg.degree
    stream = torch.cuda.current_stream()
    ctx = binding.Csf(cfg.ncell, cfg.box, cfg.order, cfg.bc, device=local, stream=stream.cuda_stream)
    if args.variant:
        ctx.set_variant(args.variant)
    t_setup = time.perf_counter()
    sysm = build_system(cfg, ctx, with_projectors=not args.no_projectors)
    M = ctx.M; rows = 2 * M
    fp32 = mode_name == "fp32"
    mode = binding.CSF_FP32_INTERMEDIATE if fp32 else binding.CSF_FP64
    wb = max(ctx.workspace_bytes(nvec, mode), ctx.workspace_bytes(nvec), ctx.rr_workspace_bytes(nvec), ctx.lanczos_workspace_bytes())
    work = torch.empty(max(wb, 16), dtype=torch.uint8, device="cuda")

    # bounds [a, b]: 20 Lanczos steps on the device (csf_lanczos) from a seeded start vector;
    # b = theta_max + |beta_k| is a safe upper bound, a = theta_min + 0.02 (b - theta_min) stands in for lambda_T (A15)
    gen0 = torch.Generator(device="cuda"); gen0.manual_seed(7)
    v0 = torch.empty((rows, 1), dtype=torch.complex128, device="cuda")
    torch.view_as_real(v0).normal_(0.0, math.sqrt(0.5), generator=gen0)
    al, be = ctx.lanczos(v0, 20, work)
    tmin, tmax = binding.tridiag_extremes(al, be)
    b = tmax + abs(float(be[-1])); a = tmin + 0.02 * (b - tmin)
    del v0

    # this rank's block of states (band group): a different seed per block index
    my_blocks = shard_states(max(cfg.nstates, nvec * world), nvec, rank, world)
    gen = torch.Generator(device="cuda"); gen.manual_seed(cfg.seed * 1000 + my_blocks[0])
    X = torch.empty((rows, nvec), dtype=torch.complex128, device="cuda")
    torch.view_as_real(X).normal_(0.0, math.sqrt(0.5), generator=gen)
    Y = torch.empty_like(X)
    t_setup = time.perf_counter() - t_setup

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        ctx.filter(X, Y, nvec, nvec, degree, a, b, mode, work)
    barrier()
    for k in range(binding.KIND_AUX + 1):
        ctx.profile_read(k)
    ctx.profile_enable(not args.no_profile)
    l0 = ctx.launch_count()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    barrier()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        ctx.filter(X, Y, nvec, nvec, degree, a, b, mode, work)
    e1.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms_local = e0.elapsed_time(e1)
    ms = reduce_max_time(ms_local, dist if world > 1 else None)
    launches = ctx.launch_count() - l0
    kinds = {binding.KIND_NAMES[k]: ctx.profile_read(k) for k in range(binding.KIND_AUX + 1)}
    ctx.profile_enable(False)
    ms_per_step = ms / steps
    units_step = float(rows) * nvec * degree
    value = world * units_step / (ms_per_step * 1e-3)
    finite = bool(torch.isfinite(torch.view_as_real(Y)).all().item())

    # ---- roofline of the dominant kernel (column kernel) and of the whole step
    rm = roofline_model(cfg.order, sysm.coverage, fp32)
    peaks = ctxs["peaks"]
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    peak64 = SM_COUNT * FP64_FMA_PER_CLK_PER_SM * 2 * sm_max * 1e6 / 1e12
    peak32 = 2.0 * peak64                                   # 128 FP32 lanes per clock and SM
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    cell_ms, cell_n = kinds["cell"]
    launch_units = float(rows) * nvec
    # time floors of one H apply (all kernels of a step): HBM, and the ALU pipes (FP32 part at the FP32 peak + FP64 part at the FP64 peak)
    t_hbm = (rm["bytes_column"] + rm["bytes_gather"]) * launch_units / (hbm * 1e9)
    t_alu = launch_units * (rm["flops_fp32"] / (peak32 * 1e12) + rm["flops_fp64"] / (peak64 * 1e12))
    roof = None
    # csf_filter's fused half-block path: every column launch works on half the block and carries, in two extra warps, the
    # projector gather of the other half (a5): its time, flops and bytes per H apply are those of two launches
    fused = (not fp32) and (not args.no_projectors) and ctx.filter_fused_gather(nvec, mode)
    per_apply = 2 if fused else 1
    f_col = rm["flops_column"] + (72.0 * sysm.coverage if fused else 0.0)
    b_col = rm["bytes_column"] + (rm["bytes_gather"] if fused else 0.0)
    if cell_n > 0:
        t_cell = cell_ms / cell_n * per_apply * 1e-3
        if fp32:
            # the column kernel's own floors: 24 B/unit, its FP32 cell flops + the FP64 expansion (72 c_ov flops/unit)
            f32c = rm["flops_column"] - 72.0 * sysm.coverage
            t_floor = max(rm["bytes_column"] * launch_units / (hbm * 1e9), launch_units * (f32c / (peak32 * 1e12) + 72.0 * sysm.coverage / (peak64 * 1e12)))
            ach = rm["flops_column"] * launch_units / t_cell / 1e12
            roof = {"kernel": "column_kernel<float> (a1-a4, a7, a8)", "bound": "alu", "achieved": ach, "peak": rm["flops_column"] * launch_units / t_floor / 1e12,
                    "unit": "TFLOP/s", "frac": t_floor / t_cell,
                    "peak_source": "mixed-pipe floor: FP32 cell flops at 148 SMs x 128 FMA/clk x 2 x %.0f MHz + FP64 expansion flops at half that, or 24 B/unit at the measured HBM copy rate, whichever is slower (DESIGN.md section 5)" % sm_max}
        else:
            ach = f_col * launch_units / t_cell / 1e12
            roof = {"kernel": "column_kernel with gather warps (a1-a5, a7, a8): two launches of half a block each per H apply" if fused else "column_kernel (a1-a4, a7, a8)",
                    "bound": "alu", "achieved": ach, "peak": peak64, "unit": "TFLOP/s", "frac": ach / peak64,
                    "peak_source": "148 SMs x 64 FP64 FMA/clk x 2 x %.0f MHz (DESIGN.md; DFMA and DMMA share these units: 36.4 TF/s measured together)" % sm_max}
        tr = ctxs["traffic"].get("cfg%d_%s%s" % (cfg.index, mode_name, "_fused" if fused else ""))
        roof.update({"traffic": (float(tr["dram_bytes_per_unit"]) * launch_units) if tr else None,
                     "traffic_source": tr["source"] if tr else None,
                     "algorithmic_bytes": b_col * launch_units, "flops_per_unit": f_col,
                     "flops_note": "algorithmic count of SURVEY 8(d) (cheapest algorithm implemented); the kernel executes fewer kinetic flops (shared z-planes are contracted once) and more projector flops (K 18 -> 20, partial row tiles)",
                     "avg_launch_ms": t_cell * 1e3 / per_apply, "launches": cell_n, "launches_per_apply": per_apply, "ms_per_apply": t_cell * 1e3,
                     "share_of_step": cell_ms / ms_local,
                     "hbm_achieved_gbs": b_col * launch_units / t_cell / 1e9, "hbm_peak_gbs": hbm,
                     "hbm_frac": b_col * launch_units / t_cell / 1e9 / hbm,
                     "hbm_peak_source": "measured (MEASURED_PEAKS.json)" if peaks else "fallback"})
    t_apply = ms_per_step * 1e-3 / degree
    step = {"flops_per_unit": rm["flops_total"], "bytes_per_unit": rm["bytes_column"] + rm["bytes_gather"],
            "floor_ms_per_apply": {"hbm": t_hbm * 1e3, "alu": t_alu * 1e3}, "ms_per_apply": t_apply * 1e3,
            "frac": max(t_hbm, t_alu) / t_apply, "frac_alu": t_alu / t_apply, "frac_hbm": t_hbm / t_apply,
            "bound": "alu" if t_alu >= t_hbm else "hbm",
            "kernel_ms": {k: round(v[0] / steps, 3) for k, v in kinds.items()}}
    conf = workload_dict(cfg, sysm)
    conf.update({"block_vectors": nvec, "degree": degree, "bounds": [a, b], "lanczos_ritz": [tmin, tmax], "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                 "mode": mode_name, "column_kernel_lanes": ctx.column_lanes(nvec, 1 if fp32 else 0), "fused_gather": bool(fused), "setup_s": round(t_setup, 2)})
    res = {"value": value, "ms_per_step": ms_per_step, "steps": steps, "warmup": warmup, "dtype": "f32" if fp32 else "f64", "config": conf, "clocks": clocks,
           "gpu_launches": launches, "roofline": roof, "step_roofline": step, "finite": finite}
    if cfg.nstates > 0:
        nblocks = math.ceil(cfg.nstates / cfg.nvec)
        res["full_filter_extrapolated_s"] = {"blocks": nblocks, "seconds": nblocks * ms_per_step * 1e-3, "note": "per-block time x blocks of the config's state count (BASELINE.json)"}
    live = {"ctx": ctx, "X": X, "Y": Y, "work": work, "a": a, "b": b, "rows": rows, "nvec": nvec, "degree": degree, "mode": mode, "barrier": barrier}
    return res, live


def measure_dense(args, peaks):
    """One H apply through csf_apply_H_dense (eq.79-84: potential at n_q^3 Gauss-Legendre points, dense cell-level
    matrices, FP64 tensor-core product) and through csf_apply_H (sum-factorised, nodal potential) on the same mesh, block and
    projectors: config 3's cell size, order and atom density on a sub-mesh whose 4 n_p^6 doubles per cell fit the GPU."""
    import torch
    from paper_2410_02754_b200 import binding
    base = synth.CONFIGS[3]
    nc = min(args.dense_cells, base.ncell[0])
    cfg = synth.scaled_config(base, (nc, nc, nc), max(1, round(base.natoms * nc ** 3 / (base.ncell[0] * base.ncell[1] * base.ncell[2]))), nvec=base.nvec)
    ctx = binding.Csf(cfg.ncell, cfg.box, cfg.order, cfg.bc)
    sysm = build_system(cfg, ctx)
    nq = cfg.order + 3
    pts = ctx.quadrature_points(nq)
    k = [2.0 * np.pi / b for b in cfg.box]
    vq = np.empty(pts.shape[:2] + (4,))
    vq[..., 0] = -1.0 + 0.5 * np.cos(k[0] * pts[..., 0]) * np.cos(k[1] * pts[..., 1]) * np.cos(k[2] * pts[..., 2])
    vq[..., 1] = 0.1 * np.sin(k[0] * pts[..., 0]); vq[..., 2] = 0.1 * np.sin(k[1] * pts[..., 1]); vq[..., 3] = 0.1 * np.cos(k[2] * pts[..., 2])
    del pts
    torch.cuda.synchronize(); t0 = time.perf_counter()
    ctx.set_potential_quadrature(nq, vq)
    ms_setup = (time.perf_counter() - t0) * 1e3
    rows, nvec = 2 * ctx.M, cfg.nvec
    gen = torch.Generator(device="cuda"); gen.manual_seed(777)
    X = torch.empty((rows, nvec), dtype=torch.complex128, device="cuda"); torch.view_as_real(X).normal_(0.0, math.sqrt(0.5), generator=gen)
    Y = torch.empty_like(X)
    work = torch.empty(max(ctx.workspace_bytes(nvec), ctx.dense_workspace_bytes(nvec), 16), dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def timed(fn, reps):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            fn()
        e1.record(stream); torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    ms_sf = timed(lambda: ctx.apply_H(X, Y, nvec, nvec, work), 5)
    ctx.profile_enable(True)
    ms_dense = timed(lambda: ctx.apply_H_dense(X, Y, nvec, nvec, work), 3)
    ms_cell, n_cell = ctx.profile_read(binding.KIND_CELL)
    rest = {binding.KIND_NAMES[kd]: (lambda r: r[0] / max(r[1], 1))(ctx.profile_read(kd)) for kd in (binding.KIND_PGATHER, binding.KIND_DELTA, binding.KIND_AUX)}
    ctx.profile_enable(False)
    # the same apply at a k-point (eq.40-42: Bloch term in the cell product, complex projectors)
    kvec = np.array([0.21, -0.13, 0.08])
    ctx.set_kpoint(kvec)
    ctx.set_projectors_complex(sysm.node_ptr, sysm.node_idx, sysm.nproj, synth.bloch_pvals(sysm, ctx.node_coords(), kvec), sysm.atom_type, sysm.delta, sysm.delta_ptr)
    ctx.set_potential_quadrature(nq, vq)
    ctx.profile_enable(True)
    ms_dense_k = timed(lambda: ctx.apply_H_dense(X, Y, nvec, nvec, work), 3)
    ms_cell_k, n_cell_k = ctx.profile_read(binding.KIND_CELL)
    ctx.profile_enable(False)
    del vq
    n3 = (cfg.order + 1) ** 3
    E = cfg.ncell[0] * cfg.ncell[1] * cfg.ncell[2]
    flops = 6.0 * 2.0 * 2.0 * n3 * n3 * nvec * E                       # six real n3 x n3 products on 2 nvec real columns per cell
    mat_bytes = 4.0 * 8.0 * n3 * n3 * E
    peak64 = SM_COUNT * FP64_FMA_PER_CLK_PER_SM * 2 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12
    ms_k = ms_cell / max(n_cell, 1)
    out = {"note": "PAPER.md eq.79-84: potential at n_q^3 Gauss-Legendre points, dense 2x2-spin cell matrix applied with FP64 tensor-core tiles; "
                   "beside it the sum-factorised csf_apply_H on the same mesh, block and projectors (nodal potential)",
           "workload": f"{cfg.name}: {cfg.ncell[0]}^3 cells, order {cfg.order}, {cfg.natoms} atoms, {nvec} vectors, n_q = {nq}",
           "cell_matrix_bytes": mat_bytes, "setup_ms": ms_setup,
           "apply_dense_ms": ms_dense, "apply_sum_factorised_ms": ms_sf, "dense_over_sum_factorised": ms_dense / ms_sf,
           "dense_kernel_ms": ms_k, "dense_kernel_tflops": flops / ms_k / 1e9, "dense_kernel_frac_of_fp64_peak": flops / ms_k / 1e9 / peak64,
           "dense_kernel_matrix_gbs_if_read_once": mat_bytes / ms_k / 1e6,
           "nonlocal_kernels_ms": {"proj_gather": rest["proj_gather"], "delta": rest["delta"], "expansion": rest["aux"]},
           "kpoint": {"k": kvec.tolist(), "apply_dense_ms": ms_dense_k, "dense_kernel_ms": ms_cell_k / max(n_cell_k, 1),
                      "dense_kernel_tflops": flops * 8.0 / 6.0 / (ms_cell_k / max(n_cell_k, 1)) / 1e9,
                      "dense_kernel_frac_of_fp64_peak": flops * 8.0 / 6.0 / (ms_cell_k / max(n_cell_k, 1)) / 1e9 / peak64,
                      "note": "eight real products per cell instead of six (the Bloch term -i k.grad), complex projector entries"},
           "units_per_s_dense": rows * nvec / (ms_dense * 1e-3), "units_per_s_sum_factorised": rows * nvec / (ms_sf * 1e-3),
           "finite": bool(torch.isfinite(torch.view_as_real(Y[::4099])).all().item())}
    del X, Y, work, ctx
    return out


def main_ours(args):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1")); rank = int(os.environ.get("RANK", "0")); local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks, traffic = {}, {}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            peaks = json.load(f)
    except OSError:
        pass
    try:
        with open(os.path.join(ROOT, "profiles", "r2_traffic.json")) as f:       # DRAM bytes per unit from one `ncu --set full` capture per (config, mode)
            traffic = json.load(f)
    except (OSError, ValueError):
        pass
    ctxs = {"world": world, "rank": rank, "local": local, "peaks": peaks, "traffic": traffic}

    head, live = measure(args.config, args.mode, args.steps, args.warmup, args, ctxs)
    if head["roofline"] is not None and not args.no_probe:
        from paper_2410_02754_b200 import binding
        pf, pm = binding.probe_fp64_peak(local)
        head["roofline"]["peak_measured_dfma"] = pf; head["roofline"]["peak_measured_dmma"] = pm
        head["roofline"]["peak_measured_dfma_and_dmma_together"] = binding.probe_fp64_mixed(local)       # = either alone: one set of FP64 units
        if args.mode == "fp64":
            head["roofline"]["frac_of_measured_dfma"] = head["roofline"]["achieved"] / pf

    ctx, X, rows, nvec, degree, a, b, mode, barrier = (live[k] for k in ("ctx", "X", "rows", "nvec", "degree", "a", "b", "mode", "barrier"))

    # ---- subspace steps after the filter: Rayleigh-Ritz on the filtered block, density
    subspace = None
    if args.mode == "fp64" and not args.no_subspace and nvec >= 2:
        from paper_2410_02754_b200 import binding
        Y, work = live["Y"], live["work"]
        stream = torch.cuda.current_stream()
        N = nvec
        dHs = torch.empty((N, N), dtype=torch.complex128, device="cuda"); dSs = torch.empty_like(dHs); dQ = torch.empty_like(dHs)
        rho = torch.empty((rows // 2, 4), dtype=torch.float64, device="cuda")
        occ = np.ones(N)

        def timed(fn, reps):
            fn(); torch.cuda.synchronize()
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                fn()
            e1.record(stream); torch.cuda.synchronize()
            return e0.elapsed_time(e1) / reps

        # the block is the filter's OUTPUT, rescaled column by column so that X^dagger X stays well conditioned
        Y.div_(Y.norm(dim=0, keepdim=True))
        ms_proj = timed(lambda: ctx.rr_project(Y, N, N, dHs, dSs, work), 2)
        t0 = time.perf_counter(); solve_err = None
        try:
            lam = ctx.rr_solve(dHs, dSs, N, dQ)
        except binding.CsfError as ex:             # (a random block filtered once can be numerically rank deficient: time the rotation with Q = I)
            solve_err = str(ex); lam = np.zeros(N); dQ.copy_(torch.eye(N, dtype=torch.complex128, device="cuda"))
        ms_solve = (time.perf_counter() - t0) * 1e3
        ms_rot = timed(lambda: ctx.rr_rotate(Y, N, N, dQ, X, N, work), 2)           # U overwrites the input block (no longer needed)
        ms_rho = timed(lambda: ctx.density(X, N, N, occ, rho), 3)
        peak64 = SM_COUNT * FP64_FMA_PER_CLK_PER_SM * 2 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12
        hbm = float(peaks.get("hbm_gbs", 6650.0))
        f_gram = 4.0 * N * N * rows                                                   # Hermitian N x N product over `rows` rows: N (N + 1) / 2 x 8 flops
        t_apply = head["ms_per_step"] / degree                                      # one H apply of the filter leg
        subspace = {"note": "Rayleigh-Ritz (PAPER.md eq.71-72) on the filtered block, density (eq.4-5); dense FP64 contractions: tensor-pipe (DMMA) bound",
                    "rr_project_ms": ms_proj, "rr_project_tflops_gemm": 2 * f_gram / max(ms_proj - t_apply, 1e-3) / 1e9,
                    "rr_project_frac_of_fp64_peak": 2 * f_gram / max(ms_proj - t_apply, 1e-3) / 1e9 / peak64,
                    "rr_solve_ms_host_wall": ms_solve, "rr_solve_error": solve_err, "ritz_min_max": [float(lam[0]), float(lam[-1])],
                    "rr_rotate_ms": ms_rot, "rr_rotate_tflops": 8.0 * N * N * rows / ms_rot / 1e9, "rr_rotate_frac_of_fp64_peak": 8.0 * N * N * rows / ms_rot / 1e9 / peak64,
                    "density_ms": ms_rho, "density_gbs": rows * N * 16.0 / ms_rho / 1e6, "density_frac_of_hbm": rows * N * 16.0 / ms_rho / 1e6 / hbm,
                    "filter_ms": head["ms_per_step"], "rr_share_of_chfsi_pass": (ms_proj + ms_solve + ms_rot) / (head["ms_per_step"] + ms_proj + ms_solve + ms_rot)}
        del dHs, dSs, dQ, rho, Y, work

    # ---- end to end: host buffers through csf_filter_host (H2D + filter + D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        import psutil
        e2e_nvec = nvec
        need = 2 * rows * 16
        avail = psutil.virtual_memory().available / max(1, world)
        while e2e_nvec > 8 and need * e2e_nvec > 0.7 * avail:
            e2e_nvec //= 2
        hX = torch.empty((rows, e2e_nvec), dtype=torch.complex128, pin_memory=True)
        if subspace is not None:                      # the block was overwritten by the rotation: draw it again
            gen = torch.Generator(device="cuda"); gen.manual_seed(4242)
            torch.view_as_real(X).normal_(0.0, math.sqrt(0.5), generator=gen)
        hX.copy_(X[:, :e2e_nvec])
        live["X"] = live["Y"] = live["work"] = None
        del X
        torch.cuda.empty_cache()
        hY = torch.empty((rows, e2e_nvec), dtype=torch.complex128, pin_memory=True)
        ctx.set_host_chunk(args.host_chunk)
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        ctx.filter_host(hX, hY, e2e_nvec, min(e2e_nvec, 2 * args.host_chunk), min(degree, 2), a, b, mode)   # warm-up: allocates both staging slots
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            ctx.filter_host(hX, hY, e2e_nvec, e2e_nvec, degree, a, b, mode)
        torch.cuda.synchronize()
        dt_ms = (time.perf_counter() - t0) * 1e3
        barrier()
        dt_ms = reduce_max_time(dt_ms, dist if world > 1 else None)
        ev = world * float(rows) * e2e_nvec * degree / (dt_ms / e2e_steps * 1e-3)
        e2e = {"value": ev, "unit": UNIT, "h2d_bytes_per_step": rows * e2e_nvec * 16, "d2h_bytes_per_step": rows * e2e_nvec * 16,
               "steps": e2e_steps, "ms_per_step": dt_ms / e2e_steps, "block_vectors": e2e_nvec, "host_chunk_columns": args.host_chunk,
               "api": "csf_filter_host (pinned host X, Y; column chunks staged H2D / filtered / D2H on three streams)",
               "finite": bool(torch.isfinite(torch.view_as_real(hY[::4097])).all().item())}
        del hX, hY
    live.clear()
    del ctx
    torch.cuda.empty_cache()

    # ---- the other roofline-target legs (BASELINE.json: configs 2-4 in complex128, config 4 also FP32-intermediate)
    others = []
    if world == 1 and not args.no_others and not (args.nvec or args.degree):
        for k, m in [(2, "fp64"), (3, "fp64"), (4, "fp64"), (4, "fp32")]:
            if (k, m) == (args.config, args.mode):
                continue
            r, lv = measure(k, m, args.other_steps, max(3, min(args.warmup, 3)), args, ctxs)
            lv.clear()
            torch.cuda.empty_cache()
            others.append({"workload": r["config"]["workload"], "mode": m, "value": r["value"], "unit": UNIT, "ms_per_step": r["ms_per_step"], "steps": r["steps"],
                           "warmup": r["warmup"], "roofline": r["roofline"], "step_roofline": r["step_roofline"], "clocks": r["clocks"], "finite": r["finite"],
                           "full_filter_extrapolated_s": r.get("full_filter_extrapolated_s"), "c_ov": r["config"].get("c_ov")})

    # ---- the paper's own form of the local part (dense cell matrices, eq.84) beside the sum-factorised one
    dense = None
    if world == 1 and not args.no_dense and not (args.nvec or args.degree):
        dense = measure_dense(args, peaks)
        torch.cuda.empty_cache()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, desc, cores, _ = run_oracle_sample(synth.CONFIGS[args.config])
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}

    if rank == 0:
        out = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": head["ms_per_step"],
               "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": head["dtype"], "data": "synthetic", "config": head["config"],
               "clocks": head["clocks"], "e2e": e2e, "gpu_launches": head["gpu_launches"], "roofline": head["roofline"], "step_roofline": head["step_roofline"],
               "cpu_baseline": cpu, "finite": head["finite"], "full_filter_extrapolated_s": head.get("full_filter_extrapolated_s"), "other_configs": others,
               "subspace": subspace, "dense_cell_matrix_path": dense}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=sorted(synth.CONFIGS))
    ap.add_argument("--nvec", type=int, default=0, help="override the block width (not a bench value)")
    ap.add_argument("--degree", type=int, default=0, help="override the degree (not a bench value)")
    ap.add_argument("--mode", default="fp64", choices=["fp64", "fp32"], help="fp32 = CSF_FP32_INTERMEDIATE (complex128 in/out, complex64 buffers)")
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--host-chunk", type=int, default=64)
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-projectors", action="store_true", help="local part only (diagnostic, not a bench value)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-profile", action="store_true")
    ap.add_argument("--no-probe", action="store_true")
    ap.add_argument("--no-subspace", action="store_true", help="skip the Rayleigh-Ritz / density timings after the headline leg")
    ap.add_argument("--no-others", action="store_true", help="skip the other roofline-target legs (configs 2, 4 in FP64, config 4 in FP32-intermediate)")
    ap.add_argument("--other-steps", type=int, default=2, help="timed steps of each other leg")
    ap.add_argument("--no-dense", action="store_true", help="skip the dense cell-matrix leg (SURVEY 8(f) NEXT-3)")
    ap.add_argument("--dense-cells", type=int, default=16, help="cells per direction of the dense leg's sub-mesh of config 3")
    args = ap.parse_args()
    return main_reference(args) if args.impl == "reference" else main_ours(args)


if __name__ == "__main__":
    sys.exit(main())

#!/usr/bin/env python
"""bench.py -- RPIM assembly throughput on B200 (quad-points/s, fp64), the BASELINE.json metric.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config stress] [--impl reference]

The headline workload is BASELINE.json configs[4] (`stress`, the largest configuration that fits one B200);
configs[3] (`large`, the other configuration north_star's target names) is timed in the same run and
reported under the extra key "large".

A "step" is one pass of the whole hot path over one synthetic
workload: rpim_build_pattern (kNN + CSR pattern) -> rpim_get_pattern -> rpim_assemble (shape functions,
B^T D B, deterministic reduction into CSR, body force) -> rpim_apply_penalty.  `value` = quadrature
points processed per second, inputs resident in HBM, timed with CUDA events on the launching stream,
max over ranks.  Extra keys give the assemble+penalty-only rate (the paper's stage 1+2, DESIGN.md
R12), the per-phase kernel times, the roofline of the dominant kernel, the end-to-end rate through
the host-buffer C ABI calls (pinned host buffers, H2D/D2H inside the timed region), and the CPU
oracle timed on a bounded sample of the same workload (a reported baseline, not the target).

N > 1 (torchrun, one rank per GPU): the path partitions (quadrature points and matrix rows are
independent per spatial partition), so every rank assembles its own partition of the
same size with no data-path collective: weak scaling, value = total points / max-over-ranks time.
With --shard the N ranks instead share ONE domain of the config (row slabs with point / node halos,
paper_1802_04256_b200/partition.py; one allreduce(max) of a double per step): strong scaling,
value = the domain's points / max-over-ranks time.

`--impl reference` times the CPU oracle (oracle/, as it stands, one host core) on bounded samples
of the same workload; under torchrun only rank 0 runs it.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import workloads  # noqa: E402

METRIC = "rpim_assembly_quad_points_per_sec"
UNIT = "quad-points/s"
FP64_LANES_PER_SM = 64            # DFMA lanes per SM per clock (4 SMSP x 16), DESIGN.md section 5
N_SM = 148


def read_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


def read_traffic(config_name: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the two hot kernels, from the committed
    `ncu --set full` summaries (profiles/traffic.csv, see profiles/traffic.md); {} when there is none."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    out = {}
    if os.path.exists(p):
        for line in open(p).read().splitlines()[1:]:
            parts = line.split(",")
            if len(parts) == 3 and parts[0] == config_name:
                out[parts[1]] = float(parts[2])
    return out


def survey_flops_per_point(k: int) -> float:
    """SURVEY.md section 8(d) work model (fma = 2, divide = 1; n = k + 4): moment build 70 k(k+1)/2, RHS 76 k,
    LU (2/3) n^3 - n^2/2, solves 8 n^2, blocks 42 k^2, accumulation 9 k^2.  115.6 k at k = 30, 521.7 k at k = 60."""
    n = k + 4
    return 70.0 * k * (k + 1) / 2 + 76.0 * k + (2.0 / 3.0) * n ** 3 - n * n / 2.0 + 8.0 * n * n + 51.0 * k * k


def flops_per_point(k: int, symmetric: bool = False):
    """Algorithmic fp64 flops per quadrature point of THIS implementation,
    fma = 2.  Returns (shape_flops, reduce_flops).  symmetric: the panel reduction accumulates the
    upper blocks only (k (k + 1) / 2 block pairs per point instead of k^2)."""
    n = k + 4
    pairs = k * (k + 1) // 2
    build = pairs * (7 + 2 * 10 + 3 + 1) + k * (6 + 2 * 10 + 3 + 5)   # t, pow (1+9 fma, 2 mul), t*P; rhs
    m = n - 8
    factor = 0
    for i in range(4):                      # 2x2 pivots: 2 fma per trailing element + multipliers
        r = n - 2 * (i + 1)
        factor += 2 * 2 * (r * (r + 1) // 2) + 5 * r + 16 * r
    factor += sum(2 * (j * (j + 1) // 2) + j + 8 * j for j in range(m))      # 1x1 pivots (+ 4 rhs)
    back = 8 * (n * (n - 1) // 2) + 8 * n
    shape = build + factor + back
    reduce_ = (k * (k + 1) // 2 if symmetric else k * k) * 18 + k * 3      # S += (w g_I) x g_J : 9 fma per block pair
    return shape, reduce_


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            parts = [p.strip() for p in r.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for nme, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": float(max(mx)) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample_rate(w, budget_s: float = 15.0):
    """CPU oracle (one core) on a bounded sample: the first S quadrature points of the workload, all
    hot-path rows (kNN, pattern, shape functions, B^T D B assembly, penalty).  Returns (points/s, S, seconds)."""
    import oracle

    def run(S):
        pts, qw = np.ascontiguousarray(w.qpts[:S]), np.ascontiguousarray(w.qw[:S])
        t0 = time.perf_counter()
        s = oracle.knn(w.nodes, pts, w.k, "grid")
        # rows touched by the sample: a contiguous node range keeps the sample's pattern small
        lo, hi = int(s.min()), int(s.max()) + 1
        sub = (s - lo).astype(np.int32)
        rp_, ci = oracle.pattern(sub, hi - lo)
        vals, f, _ = oracle.assemble(w.nodes[lo:hi], pts, qw, sub, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, rp_, ci)
        sel = (w.bc_nodes >= lo) & (w.bc_nodes < hi)
        sel[sel] = np.diff(rp_)[3 * (w.bc_nodes[sel] - lo)] > 0      # only nodes the sample touches have rows
        if sel.any():
            oracle.penalty(w.bc_nodes[sel] - lo, w.bc_mask[sel], w.bc_ubar[sel], w.penalty_alpha, True, hi - lo,
                           rp_, ci, vals, f)
        return time.perf_counter() - t0

    S = min(w.Nq, 256)
    t = run(S)
    S2 = int(min(w.Nq, max(S, S * budget_s / max(t, 1e-3))))
    if S2 > S:
        S, t = S2, run(S2)
    return S / t, S, t


def shard_workload(config_name: str, rank: int, world: int):
    """--shard: ONE domain cut into row slabs with point / node halos (paper_1802_04256_b200/partition.py, SURVEY.md
    section 8(e)): the sub-problem of rank `rank`, its Shard and the domain's total point count.  The rank's owned
    rows are complete and identical to the same rows of the undivided matrix; the only collective of a step is
    allreduce(max) of one double (the penalty's max_i K_ii)."""
    import dataclasses
    from paper_1802_04256_b200 import partition as pt
    w = workloads.config(config_name)
    sh = pt.make_shard(w.nodes, w.qpts, w.k, rank, world)
    bn, bm, bu = pt.local_bc(sh, w.bc_nodes, w.bc_mask, w.bc_ubar)
    wl = dataclasses.replace(w, nodes=np.ascontiguousarray(w.nodes[sh.node_ids]), qpts=np.ascontiguousarray(w.qpts[sh.point_ids]),
                             qw=np.ascontiguousarray(w.qw[sh.point_ids]), bc_nodes=bn, bc_mask=bm, bc_ubar=bu)
    return wl, sh, w.Nq


def rank_workload(config_name: str, rank: int, world: int):
    """The partition rank `rank` assembles.  The path shards by spatial partition (quadrature points are
    independent; K is row-partitionable) with no data-path collective: under weak scaling every
    rank gets a block of the config's size with its own jitter stream (seed + 1000 * rank)."""
    w = workloads.config(config_name)
    if world > 1 and w.meta.get("jitter", 0.0) > 0:
        nx, ny, nz = w.grid
        w = workloads.make_block(w.name, nx, ny, nz, w.h, w.meta["gauss"], w.k, w.E, w.nu, jitter=w.meta["jitter"],
                                 seed=int(w.meta.get("seed", 0)) + 1000 * rank, body=tuple(w.body), bc=w.meta["bc"],
                                 index_bits=w.index_bits)
    return w


def max_over_ranks(ms_local: float, world: int, device=None) -> float:
    """Device-timed milliseconds of this rank -> the job's time (the slowest rank's)."""
    if world <= 1:
        return float(ms_local)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def rank_allreduce(world: int, device=None):
    """allreduce(array, "min" | "max") over the ranks for partition.verify_shard (None for a single rank)."""
    if world <= 1:
        return None
    import torch
    import torch.distributed as dist

    def red(a, op):
        t = torch.from_numpy(np.ascontiguousarray(a))
        t = t.to(device) if device is not None else t
        dist.all_reduce(t, op=dist.ReduceOp.MIN if op == "min" else dist.ReduceOp.MAX)
        return t.cpu().numpy()
    return red


def check_shard(shard, w_local, support_local, nq_job: int, world: int, device=None):
    """--shard is only valid when the halo bounds every support radius on every rank and every point of the domain
    is taken by some rank (partition.py); otherwise owned rows are silently incomplete: refuse to time that."""
    from paper_1802_04256_b200 import partition as pt
    ok, missing = pt.verify_shard(shard, w_local.nodes, w_local.qpts, support_local, nq_job, rank_allreduce(world, device))
    if not ok or missing:
        raise RuntimeError(f"--shard: halo {shard.halo:.4g} is not valid for this cloud (support radius bound holds on "
                           f"every rank: {ok}; quadrature points taken by no rank: {missing}); owned rows would be "
                           "incomplete -- use a larger halo")


def job_value(points_per_rank: int, world: int, ms_step: float) -> float:
    """Whole-job throughput: the quadrature points all ranks processed per second."""
    return world * points_per_rank / (ms_step * 1e-3)


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    rates = []
    S = 0
    per_step = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for i in range(args.warmup + args.steps):
        r, S, t = oracle_sample_rate(w, budget_s=per_step)
        if i >= args.warmup:
            rates.append((S, t))
    tot_pts = sum(s for s, _ in rates)
    tot_t = sum(t for _, t in rates)
    value = tot_pts / tot_t
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{w.name} (BASELINE.json configs[{workloads.CONFIG_NAMES.index(w.name)}])",
                   "N": w.N, "Nq": w.Nq, "k": w.k},
        "sample_points_per_step": S,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": f"first {S} quadrature points per step, all hot-path rows"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def bench_config(name, args, steps, warmup, dev, rank, local_rank, world, peaks, *, do_e2e, do_solve, sample_clocks):
    """One workload through the whole hot path; returns the pieces of the JSON line."""
    import torch
    import torch.distributed as dist
    import paper_1802_04256_b200 as rp

    hbm_gbs, sm_max_mhz, peak_src = peaks
    shard = None
    nq_job = None
    if args.shard:
        w, shard, nq_job = shard_workload(name, rank, world)
    else:
        w = rank_workload(name, rank, world)
    ctx = rp.Context(local_rank)
    ctx.set_reduction({"auto": 0, "rows": 1, "panels": 2}[args.reduction])
    d_nodes = torch.from_numpy(w.nodes).to(dev)
    d_qpts = torch.from_numpy(w.qpts).to(dev)
    d_qw = torch.from_numpy(w.qw).to(dev)
    d_bcn = torch.from_numpy(w.bc_nodes).to(dev)
    d_bcm = torch.from_numpy(w.bc_mask).to(dev)
    d_bcu = torch.from_numpy(w.bc_ubar).to(dev)

    # first pass sizes the outputs (pattern is data dependent)
    if getattr(args, "index_bits", 0):
        w.index_bits = args.index_bits      # 6432 = RPIM_INDEX_MIXED: int64 row_ptr, int32 col_idx (not the default)
    nnz, bits = ctx.build_pattern(d_nodes, d_qpts, w.k, w.index_bits)
    if shard is not None:
        d_sup = torch.empty((w.Nq, w.k), dtype=torch.int32, device=dev)
        ctx.get_pattern(None, None, d_sup)
        check_shard(shard, w, d_sup.cpu().numpy(), nq_job, world, dev)
        del d_sup
    idt = torch.int32 if bits == 32 else torch.int64
    cdt = torch.int64 if bits == 64 else torch.int32
    d_rp = torch.empty(3 * w.N + 1, dtype=idt, device=dev)
    d_ci = torch.empty(nnz, dtype=cdt, device=dev)
    d_vals = torch.empty(nnz, dtype=torch.float64, device=dev)
    d_f = torch.empty(3 * w.N, dtype=torch.float64, device=dev)

    def step():
        n2, _ = ctx.build_pattern(d_nodes, d_qpts, w.k, w.index_bits)
        assert n2 == nnz
        ctx.get_pattern(d_rp, d_ci, None)
        ctx.assemble(d_qw, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, d_vals, d_f, want_singular=False)
        penalty()

    def penalty():
        if shard is None:
            ctx.apply_penalty(d_bcn, d_bcm, d_bcu, w.penalty_alpha, True, d_vals, d_f)
            return
        # sharded domain: local max_d K_dd (m = 0 applies nothing), allreduce(max) of that one double, then the
        # penalty with the absolute alpha on the owned boundary nodes
        kmax = torch.tensor([ctx.apply_penalty(None, None, None, 1.0, True, d_vals, d_f)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(kmax, op=dist.ReduceOp.MAX)
        if d_bcn.numel():
            ctx.apply_penalty(d_bcn, d_bcm, d_bcu, w.penalty_alpha * float(kmax.item()), False, d_vals, d_f)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        step()
    barrier()
    ctx.phase_totals(reset=True)
    launches0 = ctx.launch_count()
    sampler = ClockSampler(local_rank)
    if rank == 0 and sample_clocks:
        sampler.start()
    stream = torch.cuda.current_stream(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(steps):
        step()
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = ctx.launch_count() - launches0
    phase_ms, calls = ctx.phase_totals(reset=True)
    ms_step = max_over_ranks(ms_total, world, dev) / steps
    # replicas: every rank processed its own w.Nq points; sharded: the domain's points once (halo work is overhead)
    value = job_value(w.Nq, world, ms_step) if shard is None else nq_job / (ms_step * 1e-3)

    # assemble + penalty only (paper stages 1 + 2, R12), same timing discipline
    barrier()
    e0.record(stream)
    for _ in range(steps):
        ctx.assemble(d_qw, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, d_vals, d_f, want_singular=False)
        penalty()
    e1.record(stream)
    barrier()
    ms_asm = max_over_ranks(e0.elapsed_time(e1) / steps, world, dev)
    clocks = sampler.stop() if (rank == 0 and sample_clocks) else None

    # ------------------------------------------------ rooflines (live CUDA events)
    n_asm, n_pat = max(1, calls[1]), max(1, calls[0])
    kernel_ms = {"shape_functions": phase_ms[3] / n_asm, "reduce_into_csr": phase_ms[4] / n_asm,
                 "knn": phase_ms[0] / n_pat, "incidence": phase_ms[1] / n_pat, "block_pattern": phase_ms[2] / n_pat}
    kernel_ms = {kk: max_over_ranks(v, world, dev) for kk, v in kernel_ms.items()}
    shape_ms, reduce_ms = kernel_ms["shape_functions"], kernel_ms["reduce_into_csr"]
    used = {1: "rows", 2: "panels"}.get(ctx.reduction_used(), "?")
    red_params = ctx.reduction_params()
    fl_shape, fl_reduce = flops_per_point(w.k, symmetric=(used == "panels"))
    fl_survey = survey_flops_per_point(w.k)
    peak_tflops = N_SM * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    # SURVEY.md section 8(d) minimum traffic of assemble + penalty: K written once, supports, points, nodes, f
    hbm_min = nnz * 8 + w.Nq * w.k * 4 + w.Nq * 32 + w.N * 24 + 3 * w.N * 8
    staged_reread = 37 * w.Nq * w.k            # this implementation's staged gradients + incidence, read once
    traffic = read_traffic(w.name)
    reduce_name = "reduce_rows_kernel" if used == "rows" else "reduce_panels_kernel"
    t_red_alu = fl_reduce * w.Nq / (peak_tflops * 1e12) * 1e3          # ms at the FP64 peak
    t_red_hbm = hbm_min / (hbm_gbs * 1e9) * 1e3                        # ms at the HBM peak
    if reduce_ms >= shape_ms:
        if t_red_alu >= t_red_hbm:   # the kernel's own work is governed by the FP64 pipe (k = 60: 18 k^2 flops per point)
            achieved = fl_reduce * w.Nq / (reduce_ms * 1e-3) / 1e12
            roofline = {"bound": "alu", "kernel": f"{reduce_name} (reduce_into_csr)", "achieved": achieved,
                        "peak": peak_tflops, "unit": "TFLOP/s", "frac": achieved / peak_tflops,
                        "algorithmic_flops_per_launch": fl_reduce * w.Nq}
        else:
            achieved = hbm_min / (reduce_ms * 1e-3) / 1e9
            roofline = {"bound": "hbm", "kernel": f"{reduce_name} (reduce_into_csr)", "achieved": achieved,
                        "peak": hbm_gbs, "unit": "GB/s", "frac": achieved / hbm_gbs,
                        "algorithmic_bytes_per_launch": hbm_min}
        roofline["traffic"] = traffic.get(reduce_name)
        roofline["staged_reread_bytes_per_launch"] = staged_reread
    else:
        achieved = fl_shape * w.Nq / (shape_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": "shape_rows_kernel (shape_functions)", "achieved": achieved,
                    "peak": peak_tflops, "unit": "TFLOP/s", "frac": achieved / peak_tflops,
                    "traffic": traffic.get("shape_rows_kernel"),
                    "algorithmic_flops_per_launch": fl_shape * w.Nq}
    roofline["peak_source"] = (f"MEASURED_PEAKS.json hbm_gbs ({peak_src})" if roofline["bound"] == "hbm" else
                               f"derived: {N_SM} SM x {FP64_LANES_PER_SM} DFMA/clk x 2 x {sm_max_mhz:.0f} MHz "
                               "(DESIGN.md section 5); see fp64_probe")
    t_fp64_model = fl_survey * w.Nq / (peak_tflops * 1e12) * 1e3
    t_hbm_model = hbm_min / (hbm_gbs * 1e9) * 1e3
    roofline.update({
        "kernel_ms": kernel_ms,
        "shape_fp64_frac": fl_shape * w.Nq / (shape_ms * 1e-3) / 1e12 / peak_tflops,
        "reduce_fp64_frac": fl_reduce * w.Nq / (reduce_ms * 1e-3) / 1e12 / peak_tflops,
        "reduce_hbm_frac": hbm_min / (reduce_ms * 1e-3) / 1e9 / hbm_gbs,
        # the config's governing roofline, on assemble + penalty
        "config": {
            "governing": "fp64" if t_fp64_model >= t_hbm_model else "hbm",
            "assemble_penalty_ms": ms_asm,
            "flops_per_point_survey_model": fl_survey, "flops_per_point_own_count": fl_shape + fl_reduce,
            "fp64_frac_survey_model": t_fp64_model / ms_asm,
            "fp64_frac_own_count": (fl_shape + fl_reduce) * w.Nq / (ms_asm * 1e-3) / 1e12 / peak_tflops,
            "hbm_min_bytes": hbm_min, "hbm_frac": t_hbm_model / ms_asm,
            "ms_at_100pct": max(t_fp64_model, t_hbm_model), "north_star_50pct_target_ms": 2 * max(t_fp64_model, t_hbm_model),
        },
        "fp64_peak_tflops": peak_tflops, "hbm_peak_gbs": hbm_gbs, "hbm_peak_source": peak_src,
    })

    # ------------------------------------------------ moving nodes: rpim_update_nodes against a full rebuild
    update = None
    try:
        rng = np.random.default_rng(11)

        def timed_update(nodes_np):
            d_new = torch.from_numpy(np.ascontiguousarray(nodes_np)).to(dev)
            barrier()
            e0.record(stream)
            ch, rb, _ = ctx.update_nodes(d_new, None)
            e1.record(stream)
            barrier()
            return e0.elapsed_time(e1), ch, rb, d_new

        keep_ms, keep_ch, keep_rb, d_a = timed_update(w.nodes + 1e-9 * w.h * rng.uniform(-1, 1, w.nodes.shape))
        move_ms, move_ch, move_rb, d_b = timed_update(w.nodes + 1e-2 * w.h * rng.uniform(-1, 1, w.nodes.shape))
        back_ms, back_ch, back_rb, d_c = timed_update(w.nodes)          # back to the original cloud and pattern
        d_nodes = d_c
        del d_a, d_b
        update = {"api": "rpim_update_nodes", "full_build_pattern_ms": kernel_ms["knn"] + kernel_ms["incidence"] + kernel_ms["block_pattern"],
                  "move_1e-9h": {"ms": keep_ms, "changed_points": keep_ch, "pattern_rebuilt": keep_rb},
                  "move_1e-2h": {"ms": move_ms, "changed_points": move_ch, "pattern_rebuilt": move_rb},
                  "move_back": {"ms": back_ms, "changed_points": back_ch, "pattern_rebuilt": back_rb}}
    except Exception as ex:
        update = {"error": repr(ex)[:200]}

    # ------------------------------------------------ optional: stage 3 on the assembled system
    solve = None
    if do_solve:
        d_x = torch.randn(3 * w.N, dtype=torch.float64, device=dev)
        d_y = torch.empty_like(d_x)
        for _ in range(3):
            ctx.matvec(d_vals, d_x, d_y)
        barrier()
        e0.record(stream)
        for _ in range(10):
            ctx.matvec(d_vals, d_x, d_y)
        e1.record(stream)
        barrier()
        spmv_ms = e0.elapsed_time(e1) / 10
        spmv_bytes = 8 * nnz + 4 * (nnz // 9) + 2 * 8 * 3 * w.N      # values, block columns, x and y once
        d_u = torch.zeros(3 * w.N, dtype=torch.float64, device=dev)
        e0.record(stream)
        iters, rel = ctx.solve_pcg(d_vals, d_f, d_u, 1e-8, 50000)
        e1.record(stream)
        barrier()
        solve = {"spmv_ms": spmv_ms, "spmv_gbs": spmv_bytes / (spmv_ms * 1e-3) / 1e9,
                 "spmv_hbm_frac": spmv_bytes / (spmv_ms * 1e-3) / 1e9 / hbm_gbs, "spmv_algorithmic_bytes": spmv_bytes,
                 "pcg_rel_tol": 1e-8, "pcg_iters": iters, "pcg_rel_resid": rel, "pcg_ms": e0.elapsed_time(e1)}
        del d_x, d_y, d_u

    # ------------------------------------------------ end to end through the host-buffer C ABI calls
    e2e = None
    if do_e2e:
        del d_rp, d_ci, d_vals, d_f       # rpim_host_assemble owns its device buffers: make room (config 5: 125 GB)
        torch.cuda.empty_cache()
        try:
            np_idt = np.int32 if bits == 32 else np.int64
            pin = lambda a: torch.from_numpy(a).pin_memory().numpy()  # noqa: E731
            h_nodes, h_qpts, h_qw = pin(w.nodes), pin(w.qpts), pin(w.qw)
            h_bcn, h_bcm, h_bcu = pin(w.bc_nodes), pin(w.bc_mask), pin(w.bc_ubar)
            h_rp = torch.empty(3 * w.N + 1, dtype=idt, pin_memory=True).numpy()
            h_ci = torch.empty(nnz, dtype=cdt, pin_memory=True).numpy()
            h_vals = torch.empty(nnz, dtype=torch.float64, pin_memory=True).numpy()
            h_f = torch.empty(3 * w.N, dtype=torch.float64, pin_memory=True).numpy()
            assert h_rp.dtype == np_idt

            def e2e_step():
                n2, _ = ctx.host_pattern(h_nodes, h_qpts, w.k, w.index_bits)
                assert n2 == nnz
                ctx.host_assemble(h_qw, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, h_bcn, h_bcm, h_bcu,
                                  w.penalty_alpha, True, h_rp, h_ci, h_vals, h_f)

            e2e_step()
            n_e2e = max(1, min(steps, 3))
            barrier()
            e0.record(stream)
            for _ in range(n_e2e):
                e2e_step()
            e1.record(stream)
            barrier()
            ms_e2e = max_over_ranks(e0.elapsed_time(e1) / n_e2e, world, dev)
            h2d = h_nodes.nbytes + h_qpts.nbytes + h_qw.nbytes + h_bcn.nbytes + h_bcm.nbytes + h_bcu.nbytes
            d2h = h_rp.nbytes + h_ci.nbytes + h_vals.nbytes + h_f.nbytes
            e2e = {"value": world * w.Nq / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                   "d2h_bytes_per_step": int(d2h), "ms_per_step": ms_e2e, "steps": n_e2e,
                   "api": "rpim_host_pattern + rpim_host_assemble (pinned host buffers)"}
            del h_ci, h_vals
        except Exception as ex:  # report, never fake (and never a smaller workload under the same name)
            e2e = {"value": None, "unit": UNIT, "error": repr(ex)[:300]}

    out = {
        "w": w, "value": value, "ms_per_step": ms_step, "nnz": nnz, "bits": bits, "reduction": used,
        "reduction_params": red_params,
        "assemble_penalty": {"value": (world * w.Nq if shard is None else nq_job) / (ms_asm * 1e-3), "unit": UNIT, "ms_per_step": ms_asm,
                             "gdof_entries_per_s": 9.0 * w.k * w.k * (w.Nq * world if shard is None else nq_job) / (ms_asm * 1e-3) / 1e9},
        "shard": None if shard is None else {"rows": [shard.row_lo, shard.row_hi], "nodes_taken": int(shard.node_ids.size),
                                             "points_taken": int(shard.point_ids.size), "points_domain": int(nq_job), "halo": shard.halo},
        "clocks": clocks, "e2e": e2e, "launches": int(launches), "roofline": roofline, "solve": solve,
        "update_nodes": update,
    }
    try:
        out["fp64_probe"] = ctx.probe_fp64()
    except Exception as ex:
        out["fp64_probe"] = {"error": repr(ex)[:200]}
    try:
        out["fp64_dmma_probe"] = ctx.probe_fp64_dmma()
    except Exception as ex:
        out["fp64_dmma_probe"] = {"error": repr(ex)[:200]}
    ctx.close()
    torch.cuda.empty_cache()
    return out


def config_block(w, world, r):
    return {"workload": f"{w.name} (BASELINE.json configs[{workloads.CONFIG_NAMES.index(w.name)}])",
            "N": w.N, "Nq": w.Nq, "k": w.k, "nnz": r["nnz"], "index_bits": r["bits"],
            "step": "build_pattern + get_pattern + assemble + apply_penalty", "reduction": r["reduction"],
            "reduction_params": r["reduction_params"],
            "l2": "inputs and outputs larger than L2 (no flush needed)" if r["nnz"] * 8 > 2.5e8 else
                  "working set may fit L2; no flush",
            "parallelism": ("single GPU" if world == 1 and r.get("shard") is None else
                            (f"one domain sharded into {world} row slabs with point / node halos, allreduce(max) of one double "
                             "per step (partition.py)") if r.get("shard") is not None else
                            (f"{world} independent replicas of the workload, one per GPU (own jitter stream, no halo, "
                             "no collective): not a sharded assembly of one domain"))}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="stress", choices=workloads.CONFIG_NAMES)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--reduction", default="auto", choices=["auto", "rows", "panels"],
                    help="reduction kernel (rpim_set_reduction): automatic choice, row-owner, or panel")
    ap.add_argument("--shard", action="store_true",
                    help="N > 1: shard ONE domain of the config into row slabs with halos (strong scaling, allreduce(max) of "
                         "the penalty scale) instead of N independent replicas")
    ap.add_argument("--index-bits", type=int, default=0, choices=[0, 32, 64, 6432],
                    help="0: the config's own rule (BASELINE.json: 64-bit iff nnz > 2^31 - 1); 6432 = RPIM_INDEX_MIXED "
                         "(int64 row_ptr, int32 col_idx): a side measurement, never the default")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-secondary", action="store_true", help="do not also time `large` when the headline is `stress`")
    ap.add_argument("--with-solve", action="store_true",
                    help="also time stage 3 (block SpMV, block-Jacobi PCG to 1e-8) on the assembled system; extra key \"solve\"")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        args.warmup = max(args.warmup, 3) if os.environ.get("RPIM_BENCH_STRICT_WARMUP", "1") == "1" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank_workload(args.config, rank, world))
        return

    import torch
    import torch.distributed as dist

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    peaks = read_peaks()

    r = bench_config(args.config, args, args.steps, args.warmup, dev, rank, local_rank, world, peaks,
                     do_e2e=not args.no_e2e, do_solve=args.with_solve, sample_clocks=True)
    w = r["w"]
    secondary = None
    if args.config == "stress" and not args.no_secondary:
        # the other configuration BASELINE.json north_star's target names; device-timed only
        r2 = bench_config("large", args, min(args.steps, 10), 3, dev, rank, local_rank, world, peaks,
                          do_e2e=False, do_solve=False, sample_clocks=False)
        secondary = {"config": config_block(r2["w"], world, r2), "value": r2["value"], "unit": UNIT,
                     "ms_per_step": r2["ms_per_step"], "steps": min(args.steps, 10), "warmup": 3,
                     "assemble_penalty": r2["assemble_penalty"], "gpu_launches": r2["launches"],
                     "roofline": r2["roofline"], "update_nodes": r2["update_nodes"]}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        rate, S, t = oracle_sample_rate(w, budget_s=15.0)
        cpu_baseline = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": t,
                        "sample": f"first {S} quadrature points of '{w.name}', all hot-path rows (kNN, pattern, "
                                  f"shape functions, B^T D B assembly, penalty); host has {os.cpu_count()} cores"}

    if rank == 0:
        roofline = r["roofline"]
        roofline["fp64_probe"] = r["fp64_probe"]
        # scalars beside the nested records (a flat reader keeps these): measured sustained DFMA and FP64 mma.sync
        # rates on this device, and the dominant kernel's fraction of the MEASURED DFMA rate next to `frac`
        # (which stays against the derived peak, `peak_source`)
        roofline["fp64_probe_tflops"] = r["fp64_probe"].get("tflops")
        roofline["fp64_dmma_probe_tflops"] = r["fp64_dmma_probe"].get("tflops")
        if roofline.get("bound") == "alu" and roofline["fp64_probe_tflops"]:
            roofline["frac_of_measured_fp64"] = roofline["achieved"] / roofline["fp64_probe_tflops"]
        line = {
            "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
            "scaling": "strong" if args.shard else "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config_block(w, world, r),
            "assemble_penalty": r["assemble_penalty"], "clocks": r["clocks"], "e2e": r["e2e"],
            "gpu_launches": r["launches"], "roofline": roofline, "cpu_baseline": cpu_baseline,
        }
        line["update_nodes"] = r["update_nodes"]
        if r.get("shard") is not None:
            line["shard"] = r["shard"]
        if secondary is not None:
            line["large"] = secondary
        if r["solve"] is not None:
            line["solve"] = r["solve"]
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

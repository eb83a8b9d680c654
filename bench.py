#!/usr/bin/env python
"""bench.py -- throughput of the checkerboard Metropolis sweep (hpmc_sweep) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--impl reference]

A "step" is ONE hpmc_sweep(1): grid shift + cell-list build + all 2^d colour passes (every S:8(a) row) over
the whole synthetic system.  The default workload is BASELINE.json configs[2] (1 048 576 pentagons, the
"GPU-saturating size" north_star quotes the metric on); configs[1] (4096 pentagons) is timed as well and
reported under "also".  Prints ONE JSON line (rank 0).  See DESIGN.md section 8 for every definition.

N > 1: the path does not shard in this build (one GPU per system, BASELINE.json north_star) -> N independent
replicas with seeds 1..N, no data-path collective; `value` = trials of all replicas / max-over-ranks time.

--impl reference: the oracle (oracle/, serial fp64 C) timed on the host cores; see DESIGN.md section 8.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1509_04692_b200 import workloads as wl  # noqa: E402

METRIC = "trial_moves_per_sec"
UNIT = "trial moves/s"
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12      # SMs x FP32 lanes x 2 (FMA) x max SM clock
HBM_FALLBACK_GBS = 6650.0                               # B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent

# Algorithmic work per trial: the flop tariff of SURVEY.md 8(d)-F applied to the oracle's O7 work counters
# on the melted state of each state point -- candidates scanned, narrow-phase tests, separating axes per polygon test, GJK
# support calls per polyhedron test, all in early-exit serial order -- read from tests/golden/oracle_expectations.json (a data
# file written by tests/golden/make_oracle_expectations.py from the oracle alone; nothing of the oracle is executed here).
WORK_KEY = {0: "k0_disks", 1: "k1_pentagons", 2: "k1_pentagons", 3: "k3_cubes", 4: "k1_pentagons"}


def algo_flops_per_trial(k, w):
    """FMA = 2, compare/min/max = 1, RNG and integer work not counted."""
    wk = json.load(open(os.path.join(ROOT, "tests", "golden", "oracle_expectations.json")))["work"][WORK_KEY[k]]
    rot = wk["rotate_fraction"]
    gen = (1.0 - rot) * 10.0 + rot * (30.0 if w.dim == 2 else 60.0)            # trial generation
    leave = (1.0 - rot) * 4.0 * w.dim                                          # leave-cell test (translations)
    broad = (3.0 * w.dim + 2.0) * wk["candidates_scanned_per_trial"]           # subtract, dot, compare per candidate
    if w.kind == wl.KIND_DISK:
        narrow, per_test = 0.0, 0.0                                            # the broad phase is the whole test
    elif w.kind == wl.KIND_POLYGON:
        nv = w.verts.shape[0]
        axes = wk["polygon_axes_per_narrow_test"]                              # A's normals first, then B's, to the first that separates
        per_test = 14.0 * nv + (4.0 * nv + 1.0) * min(axes, nv) + (4.0 * nv + 3.0) * max(axes - nv, 0.0)
        narrow = wk["narrow_tests_per_trial"] * per_test
    else:
        nv = w.verts.shape[0]
        support = 10.0 * nv + 48.0 + 6.0 + 2.0 * nv                            # Eq. (2): two vertex scans, two rotations, argmax compares
        per_test = wk["gjk_support_calls_per_narrow_test"] * (support + 60.0)  # + simplex update per iteration
        narrow = wk["narrow_tests_per_trial"] * per_test
    return {"flops_per_trial": gen + leave + broad + narrow, "trial_generation": gen, "leave_cell": leave, "broad_phase": broad,
            "narrow_phase": narrow, "flops_per_narrow_test": per_test, "oracle_work": wk}


# ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum per colour pass of the dominant kernel, round-2 kernels
# (profiles/r2_final.md lists the captures; a dataflow / whole-sweep launch is divided by the passes it covers)
NCU_TRAFFIC = {"k2_pentagons_1M": 21.34e6 / 4, "k4_pentagons_16M": 425.0e6, "k3_cubes": 1.20e6, "k1_pentagons_4096": 0.13e6,
               "k0_disks": 0.12e6}


def state_bytes(w):
    """Bytes per particle in the cell-sorted arrays: one pose float4 in 2-D, pos + quat float4 in 3-D."""
    return 16 if w.dim == 2 else 32


def algorithmic_bytes_per_sweep(w, C, accepted_per_sweep):
    """B_sweep: build (read state + tag, keys written and read, counts + offsets, scatter) plus one
    read of all state and all cell offsets per colour pass plus the accepted write-backs."""
    S = state_bytes(w)
    ncol = 1 << w.dim
    return w.N * (2 * (S + 4) + 16 + ncol * S) + C * (12 + 4 * ncol) + S * accepted_per_sweep


def colour_pass_bytes(w, C, accepted_per_sweep):
    """Bytes one colour-pass launch must move: all state once + all cell offsets once + accepted write-backs."""
    S = state_bytes(w)
    ncol = 1 << w.dim
    return w.N * S + 4 * C + S * accepted_per_sweep / ncol


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured"
        except Exception:
            pass
    return HBM_FALLBACK_GBS, "fallback"


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled every 200 ms during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200",
                                       "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.25)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


def roofline_of(k, w, g, prof, counters, steps, total_ms, fp32_measured):
    """The roofline object of the dominant kernel (the colour pass) for one timed window: DESIGN.md section 7."""
    acc = counters["trans_acc"] + counters["rot_acc"]
    trials = counters["trials"]
    colour_ms = prof["colour_ms"] / max(prof["colour_n"], 1)
    trials_per_launch = trials / max(prof["colour_n"], 1)
    acc_per_sweep = acc / steps
    hbm, hbm_src = hbm_peak()
    work = algo_flops_per_trial(k, w)
    fp32_peak = fp32_measured if fp32_measured and fp32_measured > 0 else FP32_PEAK_TFLOPS
    bytes_launch = colour_pass_bytes(w, g.C, acc_per_sweep)
    flops_launch = work["flops_per_trial"] * trials_per_launch
    t_hbm = bytes_launch / (hbm * 1e9)
    t_alu = flops_launch / (fp32_peak * 1e12)
    if t_hbm >= t_alu:
        roof = {"bound": "hbm", "achieved": bytes_launch / (colour_ms * 1e-3) / 1e9, "peak": hbm, "unit": "GB/s",
                "peak_source": f"{hbm_src} hbm_gbs (MEASURED_PEAKS.json)"}
    else:
        roof = {"bound": "alu", "achieved": flops_launch / (colour_ms * 1e-3) / 1e12, "peak": fp32_peak, "unit": "TFLOP/s",
                "peak_source": "pure-FMA microkernel timed in this run (hpmc_measure_fp32_peak)" if fp32_measured else
                               "nominal 148 SM x 128 lanes x 2 x 1.965 GHz"}
    roof["frac"] = roof["achieved"] / roof["peak"]
    whole = prof["colour_ms"] + prof["build_ms"]
    roof.update({"traffic": NCU_TRAFFIC.get(w.name), "kernel": g.describe_pass(), "avg_launch_ms": colour_ms,
                 "avg_launch_ms_note": "per colour pass; a launch that covers several passes is counted as that many",
                 "launches_timed": prof["colour_n"], "fp32_peak_measured": fp32_measured, "fp32_peak_nominal": FP32_PEAK_TFLOPS,
                 "algorithmic_bytes_per_launch": bytes_launch, "algorithmic_flops_per_launch": flops_launch,
                 "algorithmic_flops_per_trial": work["flops_per_trial"],
                 "flops_breakdown": {q: work[q] for q in ("trial_generation", "leave_cell", "broad_phase", "narrow_phase", "flops_per_narrow_test")},
                 "oracle_work_counters": {q: work["oracle_work"][q] for q in ("sample", "candidates_scanned_per_trial", "narrow_tests_per_trial",
                                                                              "polygon_axes_per_narrow_test", "gjk_support_calls_per_narrow_test")},
                 "kernel_share_of_step": prof["colour_ms"] / total_ms, "build_share_of_step": prof["build_ms"] / total_ms,
                 "sweep_frac": max(algorithmic_bytes_per_sweep(w, g.C, acc_per_sweep) / (hbm * 1e9),
                                   work["flops_per_trial"] * trials / steps / (fp32_peak * 1e12)) / (total_ms * 1e-3 / steps),
                 "hbm_time_us": 1e6 * t_hbm, "fp32_time_us": 1e6 * t_alu, "profiled_ms_per_step": whole / steps})
    return roof


def time_gpu(w, seed, device, steps, warmup, flush, dist_ctx):
    """W untimed + K timed hpmc_sweep(1) steps on one replica; returns a dict of raw measurements."""
    import torch
    from paper_1509_04692_b200 import binding as hb
    g = hb.from_workload(w, seed=seed, device=device)
    assert g.count_overlaps() == 0, "initial state has overlaps"
    fp32_peak = g.measure_fp32_peak()              # the FP32 roofline denominator, measured on this GPU in this run
    g.sweep(w.warmup_sweeps)                       # melt the lattice (setup), untimed
    stream = g.stream
    fbuf = torch.empty(256 << 20, dtype=torch.uint8, device=device) if flush else None

    def one_step():
        if fbuf is not None:
            with torch.cuda.stream(stream):
                fbuf.add_(1)                       # 256 MiB read+write > 126 MB L2: evicts the state (on the library's stream)
        g.sweep(1)

    for _ in range(max(warmup, 3)):
        one_step()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    g.reset_counters()
    l0 = g.launch_count()
    dist_ctx.barrier(); torch.cuda.synchronize(device)
    sampler = ClockSampler(torch.device(device).index or 0) if dist_ctx.rank == 0 else None
    t_wall = time.perf_counter()
    for s, e in ev:
        if fbuf is not None:
            with torch.cuda.stream(stream):
                fbuf.add_(1)
        s.record(stream)
        g.sweep(1)
        e.record(stream)
    torch.cuda.synchronize(device); dist_ctx.barrier()
    t_wall = time.perf_counter() - t_wall
    ms = float(sum(s.elapsed_time(e) for s, e in ev))
    c = g.counters()
    launches = g.launch_count() - l0
    # the same K steps once more, now with the library's CUDA-event brackets around the build and around every colour-pass
    # launch (hpmc_set_profile): the per-kernel times of the roofline object.  Kept out of the timed window above because the
    # extra event records between the kernels cost ~5 % of a 0.23 ms step.
    g.reset_counters()
    g.set_profile(True)
    ev2 = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for s, e in ev2:
        if fbuf is not None:
            with torch.cuda.stream(stream):
                fbuf.add_(1)
        s.record(stream)
        g.sweep(1)
        e.record(stream)
    torch.cuda.synchronize(device)
    clocks = sampler.stop() if sampler else None
    prof = g.get_profile(); g.set_profile(False)
    prof["counters"] = g.counters()
    prof["ms"] = float(sum(s.elapsed_time(e) for s, e in ev2))
    assert g.count_overlaps() == 0, "overlaps after the timed window"
    return dict(g=g, ms=ms, wall_s=t_wall, counters=c, prof=prof, launches=launches, clocks=clocks, fp32_peak=fp32_peak)


def time_e2e(g, w, steps, device):
    """The same step through the host-buffer call: pinned HOST state in, one sweep, state + counters out.  2-D systems use
    hpmc_sweep_host_pose2d (one pose (x, y, qw, qz) per particle, 16 N bytes each way), 3-D systems hpmc_sweep_host (pos4 +
    quat4, 32 N bytes each way)."""
    import torch
    p, q = g.get_state()
    if w.dim == 2:
        pose = np.concatenate([p[:, :2], q[:, [0, 3]]], axis=1).astype(np.float32)
        hp = [torch.from_numpy(np.ascontiguousarray(pose)).pin_memory(), torch.empty(w.N, 4).pin_memory()]
        step = lambda cur: g.sweep_host_pose2d(hp[cur], 1, hp[1 - cur])
        nbytes, call = w.N * 16, "hpmc_sweep_host_pose2d(n=1), pinned host buffers"
    else:
        hp = [torch.from_numpy(p.copy()).pin_memory(), torch.empty(w.N, 4).pin_memory()]
        hq = [torch.from_numpy(q.copy()).pin_memory(), torch.empty(w.N, 4).pin_memory()]
        step = lambda cur: g.sweep_host(hp[cur], hq[cur], 1, hp[1 - cur], hq[1 - cur])
        nbytes, call = 2 * w.N * 16, "hpmc_sweep_host(n=1), pinned host buffers"
    step(0)                                           # warm
    g.reset_counters()
    torch.cuda.synchronize(device)
    t = time.perf_counter()
    trials = 0
    cur = 1
    for _ in range(steps):
        c = step(cur)
        cur = 1 - cur
    torch.cuda.synchronize(device)
    t = time.perf_counter() - t
    trials = c["trials"]                              # counters accumulate over the calls
    return dict(seconds=t, trials=trials, h2d=nbytes, d2h=nbytes + 56, call=call)


def sample_of(k, n_lat):
    """A smaller system at the same state point (same lattice recipe, density, shape, moves) as config k."""
    if k == 0:
        return wl.disks(n_lat)
    if k == 3:
        return wl.cubes(n_lat)
    return wl.pentagons(n_lat, name=f"pentagons_{n_lat * n_lat}_sample")


def make_oracle(ws, threads, seed=1):
    from oracle import hpmc_oracle as ho
    o = ho.Oracle(ws.dim, ws.L, ws.kind, ws.N, seed, diameter=ws.diameter, verts=ws.verts)
    o.set_moves(ws.d, ws.a, ws.n_select)
    o.set_state(ws.pos4, ws.quat4)
    o.set_threads(threads)
    return o


def timed_oracle_sweeps(o, sweeps):
    o.reset_counters()
    t = time.perf_counter()
    o.sweeps(sweeps)
    t = time.perf_counter() - t
    return o.counters()["trials"], t


def cpu_baseline(k, w):
    """The oracle as it stands (oracle/, fp64 C), timed on this box's host cores on a bounded sample of the workload: a smaller
    system at the same state point, melted first (untimed) like the GPU's, then (i) one thread -- the oracle's definition -- and
    (ii) all cores, the cells of one colour as a parallel-for (identical results)."""
    cores = os.cpu_count() or 1
    n_lat, melt, n1, nall = {0: (64, 200, 60, 300), 1: (64, 200, 60, 300), 2: (256, 50, 12, 60), 3: (12, 100, 12, 60),
                             4: (256, 10, 12, 60)}[k]
    ws = sample_of(k, n_lat)
    o = make_oracle(ws, cores)
    o.sweeps(melt)
    o.set_threads(1)
    tr1, t1 = timed_oracle_sweeps(o, n1)
    o.set_threads(cores)
    tra, ta = timed_oracle_sweeps(o, nall)
    what = f"{ws.name}: N={ws.N} at the state point of {w.name}, melted by {melt} sweeps (as the GPU run)"
    return {"value": tr1 / t1, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": t1, "sample": f"{what}; {n1} sweeps on one thread",
            "all_cores": {"value": tra / ta, "unit": UNIT, "cores": cores, "seconds": ta,
                          "sample": f"{what}; {nall} sweeps, same-colour cells as an OpenMP parallel-for over {cores} threads"},
            "host_cores_available": cores}


def run_reference(args):
    """The reference arm: the oracle as it stands on ALL host cores of the box (the cells of one colour as a parallel-for,
    results identical to the serial run), one oracle sweep per step on the config's own system -- configs 0-3 in full, config 4
    on a 1024 x 1024 sample at the same state point (a full sweep of 16.8 M particles is ~67 M fp64 trials: minutes per step)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    k = args.config
    cores = os.cpu_count() or 1
    full = wl.config(k)
    ws = full if k != 4 else sample_of(4, 1024)
    o = make_oracle(ws, cores)
    o.sweeps(args.warmup)
    trials, t = timed_oracle_sweeps(o, args.steps)
    v = trials / t
    sample = (f"{ws.name}: N={ws.N}" + ("" if k != 4 else f" at the state point of {full.name}") +
              f"; {args.steps} oracle sweeps after {args.warmup} warm-up sweeps from the lattice start; same-colour cells as an OpenMP "
              f"parallel-for over {cores} threads")
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": full.name, "N": ws.N, "same_system_as_gpu_arm": k != 4, "sample": sample},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "particle_sweeps_per_sec": ws.N * args.steps / t}
    print(json.dumps(line), flush=True)


def run_partitioned(args, D):
    """--partition: ONE system on all ranks (paper_1509_04692_b200/partition.py).  "replicated": every rank holds the whole
    state and runs the colour-pass tiles of a slab of cell rows, boundary rows after every colour and the slabs after the last
    over NCCL.  "distributed": every rank holds its slab and one ghost row, the last row of a slab is the inactive region of
    the sweep, particles are routed between neighbouring ranks once per sweep.  Same step, metric and timing rules
    as the default arm; "scaling": "strong"."""
    import torch
    from paper_1509_04692_b200 import binding as hb
    from paper_1509_04692_b200.partition import DistributedRank, DistributedState, pose_of
    device = f"cuda:{D.local}"
    torch.cuda.set_device(D.local)
    w = wl.config(args.config, seed=1)               # the SAME system and Philox seed on every rank
    assert w.dim == 2, "--partition: 2-D configs (0, 1, 2, 4)"
    g = hb.from_workload(w, seed=1, device=device)
    g.set_option("path", 2); g.set_option("flow", 0)
    assert g.count_overlaps() == 0
    g.sweep(w.warmup_sweeps)                         # melt: every rank on its own (identical trajectories)
    distributed = args.partition == "distributed"
    if not D.on:                                     # one rank: the same phase calls, nothing to exchange
        runner = None
        g.set_partition(0, 1)
    elif distributed:                                # hand every rank the melted state; it keeps its slab and ghost row
        p, q = g.get_state()
        runner = DistributedState(g, D.dist, torch.from_numpy(pose_of(p, q)).to(device), torch.arange(w.N, dtype=torch.int32, device=device))
    else:
        runner = DistributedRank(g, D.dist)

    def one_step():
        if runner is not None:
            runner.sweep(1)
        else:
            g.sweep_phase(-1)
            for ci in range(4):
                g.sweep_phase(ci)

    fbuf = torch.empty(256 << 20, dtype=torch.uint8, device=device) if not args.no_flush else None
    for _ in range(max(args.warmup, 3)):
        one_step()
    g.reset_counters()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    D.barrier(); torch.cuda.synchronize(device)
    sampler = ClockSampler(torch.device(device).index or 0) if D.rank == 0 else None
    for s, e in ev:
        if fbuf is not None:
            with torch.cuda.stream(g.stream):
                fbuf.add_(1)
        s.record(g.stream)
        one_step()
        e.record(g.stream)
    torch.cuda.synchronize(device); D.barrier()
    clocks = sampler.stop() if sampler else None
    ms = float(sum(s.elapsed_time(e) for s, e in ev))
    c = g.counters()
    t_max = D.reduce(ms * 1e-3, "MAX")
    trials_all = D.reduce(c["trials"], "SUM")        # every rank counts the trials of its own tiles
    g.set_partition(0, 1)
    assert g.count_overlaps() == 0
    if D.rank == 0:
        print(json.dumps({"metric": METRIC, "value": trials_all / t_max, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": 1e3 * t_max / args.steps, "higher_is_better": True, "scaling": "strong",
                          "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                          "config": {"workload": w.name, "N": w.N, "cells": g.C,
                                     "parallelism": (f"{args.gpus} ranks: distributed state (slab + ghost row per rank), last cell row of every "
                                                     "slab inactive during the sweep, particles routed once per sweep (NCCL)") if distributed else
                                                    (f"{args.gpus} ranks: partitioned colour passes over a replicated state, boundary rows "
                                                     "exchanged after every colour, slabs after the last (NCCL)"),
                                     "l2": "flushed between steps" if fbuf is not None else "not flushed"},
                          "particle_sweeps_per_sec": w.N * args.steps / t_max, "trials_per_step": trials_all / args.steps,
                          "gpu_launches": int(D.reduce(g.launch_count(), "SUM")), "roofline": None, "clocks": clocks}), flush=True)


def paper_states(device):
    """S:8(f)-1/2: the paper's own benchmark states, prepared by the harness (paper_1509_04692_b200/statepoints.py) and timed as
    one hpmc_sweep(n) call each; the paper's per-GPU figures (K20X, mixed precision) are quoted as context only."""
    import torch
    from paper_1509_04692_b200 import binding as hb
    from paper_1509_04692_b200 import statepoints as sp
    out = {}
    for label, make, sweeps, paper in (("pentagons_65536_phi0.676", lambda: sp.pentagons_paper_state(256, device=device), 1000,
                                        "3.89e7 trial moves/s per K20X at 65 536 per GPU (P:237)"),
                                       ("dodecahedra_110592_phi0.5", lambda: sp.dodecahedra_paper_state(48, device=device), 100,
                                        "8.16e6 trial moves/s per K20X at 131 072 per GPU (P:237-239)"),
                                       # the paper's two 3-D validation states (Table 1), lattice starts as in the paper
                                       ("spheres_131072_fcc_phi0.60", lambda: (wl.fcc_spheres(32, 0.60), (None, None)), 1000,
                                        "validation state of Table 1 (P* = 9.3135); no throughput printed"),
                                       ("trunc_octahedra_16000_bcc_phi0.7",
                                        lambda: (wl.bcc_polyhedra(wl.truncated_octahedron_vertices(0.5), 20, 0.7, a=0.15), (None, None)), 500,
                                        "validation state of Table 1 (P* = 13.8975); no throughput printed"),
                                       # rounded shapes (spheropolygons): no state point in the paper; lattice start, melted
                                       ("rounded_pentagons_65536", lambda: (wl.rounded_polygons(256), (None, None)), 1000,
                                        "spheropolygons are listed among the supported shapes (P:89); no throughput printed")):
        t0 = time.perf_counter()
        w, (acc_t, acc_r) = make()
        prep = time.perf_counter() - t0
        g = hb.from_workload(w, seed=1, device=device)
        g.sweep(200)
        g.reset_counters()
        s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(device)
        s.record(g.stream); g.sweep(sweeps); e.record(g.stream)
        torch.cuda.synchronize(device)
        ms = s.elapsed_time(e)
        c = g.counters()
        assert g.count_overlaps() == 0
        if acc_t is None:   # not tuned by the harness: report what the timed window saw
            acc_t = c["trans_acc"] / max(1, c["trans_acc"] + c["trans_rej_overlap"] + c["trans_rej_cell"])
            acc_r = c["rot_acc"] / max(1, c["rot_acc"] + c["rot_rej_overlap"])
        out[label] = {"value": c["trials"] / (ms * 1e-3), "unit": UNIT, "N": w.N,
                      "phi": w.extra.get("phi") if w.sweep_radius else sp.packing_fraction(w), "d": w.d, "a": w.a,
                      "translate_acceptance": acc_t, "rotate_acceptance": acc_r, "sweeps": sweeps, "ms_per_sweep": ms / sweeps,
                      "particle_sweeps_per_sec": w.N * sweeps / (ms * 1e-3), "kernel": g.describe_pass(), "prepared_in_s": prep,
                      "state": w.notes, "paper_context_other_hardware": paper}
        del g
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--config", type=int, default=2, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-flush", action="store_true", help="do not evict L2 between steps (L2-resident number)")
    ap.add_argument("--no-extras", action="store_true", help="skip e2e, cpu_baseline and the small-system line")
    ap.add_argument("--partition", nargs="?", const="replicated", default=None, choices=["replicated", "distributed"],
                    help="--gpus N as ONE system (strong scaling; 2-D configs; default: N replicas).  replicated: every rank holds the "
                         "whole state and runs the colour-pass tiles of its own slab of cell rows, boundary rows exchanged after every "
                         "colour.  distributed: every rank holds its slab and a ghost row, the last row of a slab is inactive during the "
                         "sweep (the paper's scheme, P:128-151), particles are routed once per sweep")
    ap.add_argument("--paper-states", action="store_true",
                    help="also prepare and time the paper's own benchmark states (65 536 pentagons at phi = 0.676 with tuned moves, "
                         "32 768 dodecahedra at phi = 0.5; P:183, P:237): about two more minutes")
    args = ap.parse_args()
    if args.impl == "reference":
        args.steps = 20 if args.steps is None else args.steps
        args.warmup = 5 if args.warmup is None else args.warmup
        run_reference(args)
        return
    args.steps = {0: 500, 1: 500, 2: 200, 3: 200, 4: 30}[args.config] if args.steps is None else args.steps
    args.warmup = {0: 50, 1: 50, 2: 20, 3: 20, 4: 5}[args.config] if args.warmup is None else args.warmup

    import torch
    from paper_1509_04692_b200 import build as hbuild
    hbuild.build()                                   # no-op when the in-tree libhpmc.so is current
    from paper_1509_04692_b200.replicas import Replicas
    D = Replicas("nccl")
    if args.partition:
        run_partitioned(args, D)
        D.close()
        return
    device = f"cuda:{D.local}"
    torch.cuda.set_device(D.local)
    k = args.config
    w = wl.config(k, seed=D.seed)                    # replica r: orientation seed and Philox seed 1 + r
    flush = not args.no_flush
    r = time_gpu(w, D.seed, device, args.steps, args.warmup, flush, D)
    g = r["g"]
    value, trials_all, t_max = D.aggregate(r["counters"]["trials"], r["ms"] * 1e-3)
    launches_all = D.reduce(r["launches"], "SUM")
    acc = r["counters"]["trans_acc"] + r["counters"]["rot_acc"]
    trials = r["counters"]["trials"]

    roof = roofline_of(k, w, g, r["prof"], r["prof"]["counters"], args.steps, r["prof"]["ms"], r["fp32_peak"])
    roof["sweep_frac"] *= r["prof"]["ms"] / r["ms"]          # whole-sweep fraction against the un-bracketed timed window
    roof["bracketed_window_ms_per_step"] = r["prof"]["ms"] / args.steps

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * t_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "cells": g.C, "n_select": w.n_select, "d": w.d, "a": w.a,
                       "step": "one hpmc_sweep(1): shift + cell list + all colour passes",
                       "melt_sweeps_before_warmup": w.warmup_sweeps,
                       "l2": "flushed between steps (256 MiB read+write)" if flush else "not flushed (state L2-resident)",
                       "parallelism": "1 gpu" if args.gpus == 1 else f"{args.gpus} independent replicas (no collective)",
                       "notes": w.notes},
            "particle_sweeps_per_sec": D.reduce(w.N, "SUM") * args.steps / t_max,
            "acceptance": acc / max(trials, 1), "trials_per_step": trials / args.steps,
            "gpu_launches": int(launches_all), "roofline": roof, "clocks": r["clocks"]}

    if not args.no_extras:
        e = time_e2e(g, w, min(args.steps, 20), device)
        e_t = D.reduce(e["seconds"], "MAX")
        e_trials = D.reduce(e["trials"], "SUM")
        line["e2e"] = {"value": e_trials / e_t, "unit": UNIT, "h2d_bytes_per_step": e["h2d"], "d2h_bytes_per_step": e["d2h"],
                       "steps": min(args.steps, 20), "call": e["call"]}
    fp32_peak_run = r["fp32_peak"]
    del g, r
    if not args.no_extras and D.rank == 0:
        if args.gpus == 1:
            line["cpu_baseline"] = cpu_baseline(k, w)
        if k == 2:
            # north_star also quotes 4096 pentagons; 65 536 pentagons is the per-GPU size of the paper's own benchmark.
            # Both are latency-bound, L2-resident by size, and timed as one hpmc_sweep(1000) call (CUDA-graph replay).
            from paper_1509_04692_b200 import binding as hb
            line["also"] = {}
            for label, wx, note in (("k1_pentagons_4096", wl.config(1), "state is 0.26 MB: resident by size"),
                                    ("pentagons_65536", wl.pentagons(256), "state is 1 MB: resident by size; the paper's K20X: 3.9e7 "
                                     "trial moves/s at this N per GPU (phi = 0.676, mixed precision; context only)")):
                gx = hb.from_workload(wx, seed=1, device=device)
                gx.sweep(200)
                gx.reset_counters()
                s, e2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize(device)
                s.record(gx.stream); gx.sweep(1000); e2.record(gx.stream)
                torch.cuda.synchronize(device)
                msx = s.elapsed_time(e2)
                cx = gx.counters()
                assert gx.count_overlaps() == 0
                # the colour-pass launches of the same system bracketed one by one (plain launches, no graph) for its roofline
                gx.reset_counters(); gx.set_profile(True)
                for _ in range(200):
                    gx.sweep(1)
                px = gx.get_profile(); gx.set_profile(False)
                rx = roofline_of(1, wx, gx, px, gx.counters(), 200, px["colour_ms"] + px["build_ms"], fp32_peak_run)
                rx["sweep_frac"] *= (px["colour_ms"] + px["build_ms"]) / 200 / (msx / 1000)     # against the graph-replay time per sweep
                line["also"][label] = {"value": cx["trials"] / (msx * 1e-3), "unit": UNIT, "sweeps": 1000, "ms_per_sweep": msx / 1000,
                                       "particle_sweeps_per_sec": wx.N * 1000 / (msx * 1e-3), "kernel": gx.describe_pass(), "l2": note,
                                       "roofline": rx}
                del gx
    if args.paper_states and D.rank == 0 and args.gpus == 1:
        line["paper_states"] = paper_states(device)
    if D.rank == 0:
        print(json.dumps(line), flush=True)
    D.close()


if __name__ == "__main__":
    main()

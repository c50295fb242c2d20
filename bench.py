#!/usr/bin/env python
"""bench.py — two-site U(1) gate updates/s (and useful FP64 GFLOP/s) of the charge-blocked MPS update on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload 3]

Workload (BASELINE.json: the metric is quoted "at chi=1024" -> configs[2]):
XXZ TEBD, M=128, d=2, N=64, chi=1024, complex128, Trotter gates exp(-i dt H_XXZ), Delta=0.5, dt=0.05, from
the Neel state.  The config's own 50 brick-wall layers are run first (untimed preparation, reported as
"trajectory"); a STEP is one further brick-wall layer (2 columns = M-1 = 127 two-site updates, every
step a1-a5 of the hot path) on that saturated state, so that every timed step does the same, maximal work.
The state touched by a step (~M chi^2 x 16 B >> 126 MB) is larger than L2, so no explicit flush is needed.

`value`  : gates/s with gates and state resident in HBM (device gate pointers, no readback).
`e2e`    : same layers through the same C-ABI call with HOST gate buffers (pinned; copied H2D inside the call)
           plus the a6 readout of the step (<n_k>, S_k, log-norm) copied D2H, all inside the timed region.
`roofline`: dominant kernel (a3 batched Jacobi SVD), bound "alu" (FP64 pipe): useful SVD flops of the launches
           in the timed region / their summed CUDA-event durations (events recorded by the library on its stream).
`cpu_baseline` / `--impl reference`: the numpy oracle (oracle/u1mps_oracle.py, as it stands) timed on this box's host
           cores on a bounded sample: gates on seeded synthetic saturated-bond states with the sector profile of
           this workload (inputs.synthetic_gate_state; the oracle cannot reach layer 50 in minutes).
N > 1: the path does not shard (north_star: one GPU) -> N independent replicas, one per rank, no collective in
the data path ("replicas only", scaling "weak"); time = max over ranks.
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import math
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2303_11409_b200 import inputs  # noqa: E402  (seeded input generators only)

# FP64 peak used as the "alu" roofline denominator: 148 SMs x 64 FP64 FMA/clk/SM x 2 flop
# x 1.965 GHz (clocks.max.sm of MEASURED_PEAKS.json).  MEASURED_PEAKS.json has no FP64 entry; the probe result is in DESIGN.md.
FP64_FMA_PER_CLK_PER_SM = 64
SYNTH_R = {2: 9, 3: 11, 4: 13, 5: 21}   # number of charge sectors of a saturated bond (DESIGN.md §Input recipe)


def fp64_peak_tflops():
    sms, mhz = 148, 1965.0
    try:
        mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        mhz = float(mp.get("sm_max_mhz", mhz))
    except Exception:
        pass
    return sms * FP64_FMA_PER_CLK_PER_SM * 2 * mhz * 1e6 / 1e12


# ----------------------------------------------------------------------------- flop / byte accounting (host, integers)
def gate_work(d, N, tabL, tabC, tabR):
    """Algorithmic work of one gate from the three bond tables {c: n}:
    a2 flops (minimum form), useful a3 flops, bytes read+written of the two Gammas."""
    a2 = 0
    for cl, nl in tabL.items():
        for cr, nr in tabR.items():
            if not (0 <= cl - cr <= 2 * (d - 1)):
                continue
            for cp, nc in tabC.items():
                if 0 <= cl - cp <= d - 1 and 0 <= cp - cr <= d - 1:
                    a2 += 8 * nl * nc * nr
    a3 = 0
    blocks = []
    for c in range(N + 1):
        rows = sum(tabL.get(c + i, 0) for i in range(d))
        cols = sum(tabR.get(c - j, 0) for j in range(d))
        if rows == 0 or cols == 0:
            continue
        m, n = max(rows, cols), min(rows, cols)
        a3 += 4 * min(14 * m * n * n + 8 * n ** 3, 6 * m * n * n + 20 * n ** 3)
        blocks.append((m, n))
    by = 0
    for cl, nl in tabL.items():
        for i in range(d):
            by += 2 * 16 * nl * tabC.get(cl - i, 0)
    for cp, nc in tabC.items():
        for j in range(d):
            by += 2 * 16 * nc * tabR.get(cp - j, 0)
    return a2, a3, by, blocks


def layer_work(gpu, w):
    tabs = [dict(gpu.bond_info(k)) for k in range(w.M + 1)]
    a2 = a3 = by = 0
    nblk, maxblk = 0, (0, 0)
    for t in (0, 1):
        for s in inputs.column_sites(w.M, t):
            x2, x3, b, blocks = gate_work(w.d, w.N, tabs[s], tabs[s + 1], tabs[s + 2])
            a2 += x2; a3 += x3; by += b
            nblk += len(blocks)
            if blocks:
                maxblk = max(maxblk, max(blocks))
    dims = [sum(t.values()) for t in tabs]
    return {"a2_flops": a2, "a3_flops": a3, "gamma_bytes": by, "svd_blocks": nblk, "max_block": list(maxblk),
            "bond_dim_max": max(dims), "bond_dim_median": int(statistics.median(dims)),
            "sectors_max": max(len(t) for t in tabs)}


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out, _ = self.p.communicate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        busy = [x for x in sm if x > 0.5 * max(sm)] or sm
        return {"sm_mhz": statistics.median(busy), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


# ----------------------------------------------------------------------------- the oracle leg (host cores)
def oracle_sample(w, n_gates, seed0=4242):
    """Time the oracle, as it stands, on n_gates seeded synthetic saturated-bond gates of workload w.
    Returns (gates/s, seconds, cores)."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    from u1mps_oracle import U1MPS as Oracle   # the ONLY use of oracle/ here: the timed CPU baseline
    rng = np.random.default_rng(w.seed)
    cols = list(inputs.gate_columns(w, 1))
    total = 0.0
    for g in range(n_gates):
        M, N, s, lam, gam = inputs.synthetic_gate_state(w.d, w.chi, SYNTH_R[w.index], seed=seed0 + g,
                                                        profile=inputs.SATURATED_PROFILE.get(w.index))
        occ, left = [0] * M, N
        for i in range(M):
            occ[i] = min(w.d - 1, left)
            left -= occ[i]
        ora = Oracle.product_state(M, w.d, N, w.chi, occ)
        for k in (2, 3, 4):
            ora.sectors[k] = sorted(lam[k])
            ora.lam[k] = lam[k]
        for st in (2, 3):
            ora.gam[st] = gam[st]
        U = cols[0][1][g % len(cols[0][1])]
        t0 = time.perf_counter()
        ora.apply_gate(s, U, chi=w.chi, cutoff=w.cutoff)
        total += time.perf_counter() - t0
    try:
        from threadpoolctl import threadpool_info
        cores = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        cores = os.cpu_count() or 1
    return n_gates / total, total, cores


def sample_profile(w):
    prof = inputs.SATURATED_PROFILE.get(w.index)
    if prof is not None:
        return f"sector sizes {list(prof)} as measured on this workload's trajectory after {w.columns} columns"
    return f"{SYNTH_R[w.index]} sectors, parabolic profile"


def dist_max(values, world, device):
    """Max over ranks of a list of floats (the timed regions); a plain identity for world == 1.
    Used with NCCL tensors by the GPU arm and with gloo/CPU tensors by tests/test_bench_contract.py."""
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def memory_stages(prof, work, work_after, steps):
    """Achieved GB/s of the memory-bound a5 scatter: algorithmic bytes (read V, W out of the workspace + write the two
    new Gammas = the Gamma bytes of the layer) / its summed CUDA-event time; against the measured
    copy bandwidth of MEASURED_PEAKS.json.  At chi <= 1024 the per-gate working set is L2-resident."""
    ms, n = prof.get("a5_scatter", (0.0, 0))
    if ms <= 0:
        return None
    by = 0.5 * (work["gamma_bytes"] + work_after["gamma_bytes"]) * steps
    hbm = None
    try:
        hbm = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        pass
    gbs = by / (ms * 1e-3) / 1e9
    return {"a5_scatter": {"achieved": gbs, "unit": "GB/s", "peak": hbm, "frac": (gbs / hbm) if hbm else None,
                           "bytes_per_step": by / steps, "ms_per_step": ms / steps}}


def svd_traffic_bytes():
    """DRAM bytes (read + write) of ONE a3 launch from the committed ncu --set full capture, or None."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "svd_traffic.csv")) as f:
            row = next(csv.DictReader(f))
        return float(row["dram_bytes_read"]) + float(row["dram_bytes_write"])
    except Exception:
        return None


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    sample_gates = args.ref_gates
    for _ in range(args.warmup):
        oracle_sample(w, 1)
    t_tot, n_tot, cores = 0.0, 0, 1
    for k in range(args.steps):
        rate, secs, cores = oracle_sample(w, sample_gates, seed0=4242 + 1000 * k)
        t_tot += secs
        n_tot += sample_gates
    val = n_tot / t_tot
    sample = (f"{sample_gates} gates/step on seeded synthetic saturated-bond states (d={w.d}, chi={w.chi}, "
              f"{sample_profile(w)}), numpy oracle")
    print(json.dumps({
        "impl": "reference", "metric": "two-site U(1) gate updates/sec", "value": val, "unit": "gates/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "c128", "data": "synthetic",
        "config": {"workload": w.name, "M": w.M, "d": w.d, "N": w.N, "chi": w.chi, "step": sample},
        "cpu_baseline": {"value": val, "unit": "gates/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "gates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ----------------------------------------------------------------------------- our arm
def run_ours(args, w):
    import torch
    import torch.distributed as dist
    from paper_2303_11409_b200.binding import U1MPS

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # arena: state + plan + workspace for a whole column of saturated gates
    Gcol = w.M // 2
    ws_gate = 2 * w.d * w.chi * w.chi * 16
    from paper_2303_11409_b200.binding import load_library
    need = load_library().u1mps_workspace_bytes(w.M, w.d, w.N, w.chi)
    free, _ = torch.cuda.mem_get_info()
    arena = min(need + Gcol * ws_gate, int(free * 0.8))
    gpu = U1MPS(w.M, w.d, w.N, w.chi, arena_bytes=arena)
    gpu.set_product_state(w.occ)

    cols_per_layer = 2
    n_prep = w.columns if args.prep_columns < 0 else args.prep_columns
    n_total = n_prep + cols_per_layer * (args.warmup + args.steps) * 2 + cols_per_layer
    host_cols = list(inputs.gate_columns(dataclasses.replace(w, columns=n_total)))
    dev_cols = [(s, torch.from_numpy(u).cuda()) for s, u in host_cols]
    pin_cols = []
    for s, u in host_cols:
        t = torch.from_numpy(u).pin_memory()
        pin_cols.append((s, t))
    col = 0

    # ---- preparation: the config's own trajectory (untimed for the metric; reported)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(n_prep):
        gpu.apply_gate_column(dev_cols[col][0], dev_cols[col][1], cutoff=w.cutoff)
        col += 1
    e1.record()
    torch.cuda.synchronize()
    prep_ms = e0.elapsed_time(e1)
    prep_gates = sum(len(host_cols[c][0]) for c in range(n_prep))
    stats_prep = gpu.last_stats()
    work = layer_work(gpu, w)
    gates_per_step = sum(len(inputs.column_sites(w.M, t)) for t in (0, 1))

    def layer(cols_src):
        nonlocal col
        for _ in range(cols_per_layer):
            gpu.apply_gate_column(cols_src[col][0], cols_src[col][1], cutoff=w.cutoff)
            col += 1

    # ---- device-resident timed region
    for _ in range(args.warmup):
        layer(dev_cols)
    sampler = ClockSampler(local) if rank == 0 else None
    gpu.profile_enable(True)
    l0 = gpu.launch_count()
    barrier()
    e0.record()
    for _ in range(args.steps):
        layer(dev_cols)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = gpu.launch_count() - l0
    prof = gpu.profile_read()
    gpu.profile_enable(False)
    clocks = sampler.stop() if sampler else None
    work_after = layer_work(gpu, w)

    # ---- end-to-end timed region: host gate buffers in, readouts out
    for _ in range(min(args.warmup, 1)):
        layer(pin_cols)
        gpu.expect_n_all(); gpu.bond_entropy_all(); gpu.log_norm()
    barrier()
    e0.record()
    for _ in range(args.steps):
        layer(pin_cols)
        n_k = gpu.expect_n_all()
        s_k = gpu.bond_entropy_all()
        ln = gpu.log_norm()
    e1.record()
    barrier()
    ms_e2e = e0.elapsed_time(e1)
    h2d = gates_per_step * (w.d ** 4) * 16 + gates_per_step * 4
    d2h = (w.M + (w.M + 1) + 1) * 8 + 3 * 4
    stats = gpu.last_stats()
    total_n = float(np.sum(n_k))

    ms, ms_e2e = dist_max([ms, ms_e2e], world, "cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    n_gates = args.steps * gates_per_step * world
    value = n_gates / (ms * 1e-3)
    e2e = n_gates / (ms_e2e * 1e-3)
    svd_ms, svd_n = prof["a3_svd"]
    peak = fp64_peak_tflops()
    a3_flops_launch = 0.5 * (work["a3_flops"] + work_after["a3_flops"]) / cols_per_layer   # per column = per launch
    achieved = a3_flops_launch / (svd_ms / max(svd_n, 1) * 1e-3) / 1e12 if svd_ms > 0 else 0.0
    useful_flops_step = 0.5 * (work["a2_flops"] + work["a3_flops"] + work_after["a2_flops"] + work_after["a3_flops"])
    stage_ms = {k: round(v[0] / args.steps, 4) for k, v in prof.items()}

    # ---- the oracle timed beside it (rank 0, N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        rate, secs, cores = oracle_sample(w, args.cpu_gates)
        cpu = {"value": rate, "unit": "gates/s", "cores": cores, "kind": "oracle",
               "sample": f"{args.cpu_gates} gates on seeded synthetic saturated-bond states (d={w.d}, chi={w.chi}, "
                         f"{sample_profile(w)}), {secs:.1f} s of numpy/LAPACK work"}

    out = {
        "metric": "two-site U(1) gate updates/sec", "value": value, "unit": "gates/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "c128", "data": "synthetic",
        "config": {"workload": w.name, "M": w.M, "d": w.d, "N": w.N, "chi": w.chi, "cutoff": w.cutoff,
                   "step": f"one brick-wall layer ({gates_per_step} gates, 2 launches of every kernel) on the state after "
                           f"{n_prep} columns of the config's trajectory",
                   "l2": "state touched per step exceeds L2 (inputs larger than L2, no flush)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "bond_dim_max": work["bond_dim_max"], "bond_dim_median": work["bond_dim_median"],
                   "sectors_max": work["sectors_max"], "svd_blocks_per_step": work["svd_blocks"],
                   "max_block": work["max_block"]},
        "e2e": {"value": e2e, "unit": "gates/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": ms_e2e / args.steps},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": {"kernel": "svd_kernel (a3)", "bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                     "frac": achieved / peak, "traffic": svd_traffic_bytes(),
                     "peak_source": "derived: 148 SMs x 64 FP64 FMA/clk x 2 x sm_max_mhz (no FP64 entry in MEASURED_PEAKS.json; "
                                    "the round-1 probe measured 36.8 DFMA / 37.06 DMMA TFLOP/s, DESIGN.md section 6)",
                     "traffic_source": "profiles/svd_traffic.csv (ncu --set full, one launch of the same workload)",
                     "flops": "useful SVD flops 4*min(14mn^2+8n^3, 6mn^2+20n^3) per block (SURVEY §8(d))",
                     "ms_per_launch": svd_ms / max(svd_n, 1), "launches": svd_n,
                     "share_of_step": svd_ms / ms if ms > 0 else None},
        "useful_gflops": useful_flops_step * args.steps * world / (ms * 1e-3) / 1e9,
        "memory_bound_stages": memory_stages(prof, work, work_after, args.steps),
        "a2_contract": {"useful_tflops": (0.5 * (work["a2_flops"] + work_after["a2_flops"]) * args.steps
                                          / (prof["a2_contract"][0] * 1e-3) / 1e12) if prof["a2_contract"][0] > 0 else None,
                        "note": "minimum-form flops 8 nL nC nR per (c_l, c', c_r) triple / summed CUDA-event time of contract_kernel"},
        "useful_frac_of_fp64_peak": useful_flops_step * args.steps * world / (ms * 1e-3) / 1e12 / (peak * world),
        "stage_ms_per_step": stage_ms,
        "trajectory": {"gates": prep_gates, "ms": prep_ms, "gates_per_s": prep_gates / (prep_ms * 1e-3) if prep_ms > 0 else None},
        "state": {"sum_n": total_n, "log_norm": ln, "discarded": stats["discarded"], "svd_sweeps_max": stats["sweeps"],
                  "svd_converged": stats["converged"]},
        "cpu_baseline": cpu,
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=4)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", type=int, default=3, help="BASELINE.json config index (1-based); 3 = chi=1024")
    ap.add_argument("--prep-columns", type=int, default=-1, help="columns run before timing (-1: the config's own)")
    ap.add_argument("--cpu-gates", type=int, default=96, help="oracle gates in the cpu_baseline sample")
    ap.add_argument("--ref-gates", type=int, default=8, help="oracle gates per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    w = inputs.WORKLOADS[args.workload]
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()

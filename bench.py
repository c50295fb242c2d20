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
SYNTH_R = {1: 4, 2: 9, 3: 11, 4: 13, 5: 21}   # number of charge sectors of a saturated bond (DESIGN.md §Input recipe)


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
def fp64_probe():
    """Measured DFMA / DMMA throughput of this GPU (paper_2303_11409_b200/csrc/fp64_probe.cu, built by build())."""
    exe = os.path.join(ROOT, "paper_2303_11409_b200", "fp64_probe")
    try:
        out = subprocess.run([exe], capture_output=True, text=True, timeout=60).stdout.strip().splitlines()[-1]
        return json.loads(out)
    except Exception as e:  # the probe is a report, not a dependency of the measurement
        return {"error": f"{type(e).__name__}: {e}"}


def readout_bytes(gpu, w):
    """Algorithmic bytes of one a6 read-out of the whole chain: <n_k> reads every Gamma block with occupation >= 1 once
    (16 B per element) and the lambda vectors of its two bonds; the entropies read every lambda once."""
    tabs = [dict(gpu.bond_info(k)) for k in range(w.M + 1)]
    by = 0
    for s in range(w.M):
        for cl, nl in tabs[s].items():
            for i in range(1, w.d):
                by += 16 * nl * tabs[s + 1].get(cl - i, 0)
        by += 8 * (sum(tabs[s].values()) + sum(tabs[s + 1].values()))
    by += 8 * sum(sum(t.values()) for t in tabs)
    return by


def env_flops(gpu, w):
    """Useful flops of one u1mps_expect_n_full call: per site the five grouped complex GEMMs of csrc/envs.cu (E Gamma;
    the same weighted by the occupation, for blocks with i >= 1; Gamma^H T; Gamma lam R lam; S Gamma^H), 8 real flops per
    complex multiply-add, over the (cl, cr) blocks of the current sector tables."""
    tabs = [dict(gpu.bond_info(k)) for k in range(w.M + 1)]
    fl = 0
    for s in range(w.M):
        for cl, nl in tabs[s].items():
            for i in range(w.d):
                nr = tabs[s + 1].get(cl - i, 0)
                if nr:
                    fl += 8 * (nl * nl * nr * (2 if i else 1) + nr * nr * nl + nl * nr * nr + nl * nl * nr)
    return fl


def measure(w, args, steps, warmup, prep_columns, with_e2e, rank, world, local, barrier):
    """One workload on this rank's GPU: the config's own columns as preparation, then `steps` timed brick-wall layers."""
    import torch
    from paper_2303_11409_b200.binding import U1MPS, load_library
    Gcol = w.M // 2
    ws_gate = 2 * w.d * w.chi * w.chi * 16
    need = load_library().u1mps_workspace_bytes(w.M, w.d, w.N, w.chi)
    free, _ = torch.cuda.mem_get_info()
    arena = min(need + Gcol * ws_gate, int(free * 0.8))
    gpu = U1MPS(w.M, w.d, w.N, w.chi, arena_bytes=arena)
    gpu.set_product_state(w.occ)

    cols_per_layer = 2
    n_prep = w.columns if prep_columns < 0 else prep_columns
    n_total = n_prep + cols_per_layer * (warmup + steps) * (2 if with_e2e else 1) + cols_per_layer
    host_cols = list(inputs.gate_columns(dataclasses.replace(w, columns=n_total)))
    dev_cols = [(s, torch.from_numpy(u).cuda()) for s, u in host_cols]
    pin_cols = [(s, torch.from_numpy(u).pin_memory()) for s, u in host_cols] if with_e2e else None
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
    work = layer_work(gpu, w)
    gates_per_step = sum(len(inputs.column_sites(w.M, t)) for t in (0, 1))

    def layer(cols_src):
        nonlocal col
        for _ in range(cols_per_layer):
            gpu.apply_gate_column(cols_src[col][0], cols_src[col][1], cutoff=w.cutoff)
            col += 1

    # ---- device-resident timed region
    for _ in range(warmup):
        layer(dev_cols)
    sampler = ClockSampler(local) if (rank == 0 and with_e2e) else None
    gpu.profile_enable(True)
    l0 = gpu.launch_count()
    barrier()
    e0.record()
    for _ in range(steps):
        layer(dev_cols)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = gpu.launch_count() - l0
    prof = gpu.profile_read()
    clocks = sampler.stop() if sampler else None
    work_after = layer_work(gpu, w)

    # ---- end-to-end timed region: host gate buffers in, readouts out (per-kernel events stay on: a6 is timed here)
    ms_e2e = None
    a6 = None
    n_k = gpu.expect_n_all()
    ln = gpu.log_norm(allow_nonconverged=True)
    if with_e2e:
        for _ in range(min(warmup, 1)):
            layer(pin_cols)
            gpu.expect_n_all(); gpu.bond_entropy_all(); gpu.log_norm(allow_nonconverged=True)
        gpu.profile_read()
        barrier()
        e0.record()
        for _ in range(steps):
            layer(pin_cols)
            n_k = gpu.expect_n_all()
            s_k = gpu.bond_entropy_all()
            ln = gpu.log_norm(allow_nonconverged=True)
        e1.record()
        barrier()
        ms_e2e = e0.elapsed_time(e1)
        a6_ms, a6_n = gpu.profile_read()["a6_readout"]
        a6 = {"ms_per_step": a6_ms / steps, "launches_per_step": a6_n / steps, "bytes_per_step": readout_bytes(gpu, w)}
    gpu.profile_enable(False)
    stats = gpu.last_stats()
    full = None
    if with_e2e:   # full-environment read-out (exact after truncation): sum_k <n_k> = N is the check, timed once
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        n_full = gpu.expect_n_full()
        full = {"sum_n_full": float(np.sum(n_full)), "max_abs_diff_to_canonical": float(np.max(np.abs(n_full - n_k))),
                "seconds": time.perf_counter() - t0}
        full["useful_tflops"] = env_flops(gpu, w) / full["seconds"] / 1e12   # wall clock of the whole call (table read-back,
        full["note"] = "useful_tflops = five grouped complex128 GEMMs per site / wall time of the call"   # uploads, sync)
    fock = None
    if with_e2e:   # Fock-pattern sampling: 256 patterns from seeded uniform numbers, timed once
        u = np.random.default_rng(20230311).random((256, w.M))
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        pat, logp = gpu.sample_fock(u)
        fock = {"samples": 256, "seconds": time.perf_counter() - t0, "all_patterns_conserve_N": bool(np.all(pat.sum(axis=1) == w.N)),
                "mean_log_prob": float(np.mean(logp)), "distinct_patterns": int(len({bytes(r) for r in pat}))}
    res = {"w": w, "ms": ms, "ms_e2e": ms_e2e, "launches": launches, "prof": prof, "clocks": clocks, "work": work,
           "work_after": work_after, "gates_per_step": gates_per_step, "prep_ms": prep_ms, "prep_gates": prep_gates,
           "n_prep": n_prep, "stats": stats, "sum_n": float(np.sum(n_k)), "log_norm": ln, "a6": a6, "steps": steps, "full": full, "fock": fock}
    gpu.close()
    del gpu, dev_cols, pin_cols
    torch.cuda.empty_cache()
    return res


def a3_roofline(res, peak):
    """Useful FP64 rate of the a3 launches of a measurement against the FP64 peak."""
    svd_ms, svd_n = res["prof"]["a3_svd"]
    per_launch = 0.5 * (res["work"]["a3_flops"] + res["work_after"]["a3_flops"]) / 2   # per column = per launch
    achieved = per_launch / (svd_ms / max(svd_n, 1) * 1e-3) / 1e12 if svd_ms > 0 else 0.0
    return achieved, achieved / peak, svd_ms / max(svd_n, 1), svd_n


def hbm_peak():
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        return None


def svd_traffic_bytes(name):
    """DRAM bytes (read + write) of ONE a3 launch from the committed ncu --set full capture of THIS workload, or None."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", f"svd_traffic_{name}.csv")) as f:
            row = next(csv.DictReader(f))
        return float(row["dram_bytes_read"]) + float(row["dram_bytes_write"])
    except Exception:
        return None


# per-workload side measurements of the default run: (prep columns, warm-up steps, timed steps, oracle gates)
SIDE = {1: (-1, 3, 4, 64), 2: (-1, 3, 3, 32), 3: (-1, 3, 3, 24), 4: (-1, 3, 3, 8), 5: (12, 0, 1, 1)}


def run_ours(args, w):
    import torch
    import torch.distributed as dist

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

    probe = fp64_probe() if rank == 0 else None
    res = measure(w, args, args.steps, args.warmup, args.prep_columns, True, rank, world, local, barrier)
    ms, ms_e2e = dist_max([res["ms"], res["ms_e2e"]], world, "cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    gates_per_step = res["gates_per_step"]
    work, work_after, prof, stats = res["work"], res["work_after"], res["prof"], res["stats"]
    n_gates = args.steps * gates_per_step * world
    value = n_gates / (ms * 1e-3)
    e2e = n_gates / (ms_e2e * 1e-3)
    h2d = gates_per_step * (w.d ** 4) * 16 + gates_per_step * 4
    d2h = (w.M + (w.M + 1) + 1) * 8 + 3 * 4
    peak = fp64_peak_tflops()
    achieved, frac, ms_launch, svd_n = a3_roofline(res, peak)
    svd_ms = prof["a3_svd"][0]
    useful_flops_step = 0.5 * (work["a2_flops"] + work["a3_flops"] + work_after["a2_flops"] + work_after["a3_flops"])
    stage_ms = {k: round(v[0] / args.steps, 4) for k, v in prof.items()}
    stage_ms["a6_readout"] = round(res["a6"]["ms_per_step"], 4)   # timed in the end-to-end region (the device-resident one reads nothing)
    mem = memory_stages(prof, work, work_after, args.steps) or {}
    hbm = hbm_peak()
    if res["a6"]["ms_per_step"] > 0:
        gbs = res["a6"]["bytes_per_step"] / (res["a6"]["ms_per_step"] * 1e-3) / 1e9
        mem["a6_readout"] = {"achieved": gbs, "unit": "GB/s", "peak": hbm, "frac": (gbs / hbm) if hbm else None,
                             "bytes_per_step": res["a6"]["bytes_per_step"], "ms_per_step": res["a6"]["ms_per_step"],
                             "note": "<n_k> of all sites + all bond entropies once per step, CUDA-event time of the a6 kernels"}

    # ---- the oracle timed beside it (rank 0, N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        rate, secs, cores = oracle_sample(w, args.cpu_gates)
        cpu = {"value": rate, "unit": "gates/s", "cores": cores, "kind": "oracle",
               "sample": f"{args.cpu_gates} gates on seeded synthetic saturated-bond states (d={w.d}, chi={w.chi}, "
                         f"{sample_profile(w)}), {secs:.1f} s of numpy/LAPACK work"}

    # ---- the other workloads of BASELINE.json, shorter (rank 0, N = 1 only): gates/s, a3 roofline fraction, oracle beside it
    per_workload = None
    if world == 1 and not args.no_per_workload:
        per_workload = {}
        for idx in sorted(inputs.WORKLOADS):
            wi = inputs.WORKLOADS[idx]
            if idx == w.index:
                per_workload[wi.name] = {"gates_per_s": value, "a3_frac_of_fp64_peak": frac, "svd_sweeps_max": stats["sweeps"],
                                         "cpu_baseline_gates_per_s": cpu["value"] if cpu else None, "note": "the headline measurement above"}
                continue
            prep, wu, st_, og = SIDE[idx]
            r = measure(wi, args, st_, wu, prep, False, 0, 1, local, barrier)
            ach, fr, msl, _ = a3_roofline(r, peak)
            entry = {"gates_per_s": st_ * r["gates_per_step"] / (r["ms"] * 1e-3), "ms_per_step": r["ms"] / st_, "steps": st_, "warmup": wu,
                     "prep_columns": r["n_prep"], "trajectory_gates_per_s": r["prep_gates"] / (r["prep_ms"] * 1e-3) if r["prep_ms"] > 0 else None,
                     "a3_useful_tflops": ach, "a3_frac_of_fp64_peak": fr, "a3_ms_per_launch": msl,
                     "a3_share_of_step": r["prof"]["a3_svd"][0] / r["ms"] if r["ms"] > 0 else None,
                     "svd_sweeps_max": r["stats"]["sweeps"], "svd_converged": r["stats"]["converged"],
                     "bond_dim_max": r["work"]["bond_dim_max"], "max_block": r["work"]["max_block"], "sum_n": r["sum_n"]}
            if idx == 5:
                entry["note"] = ("bounded: state after the first 12 of the config's 100 columns (47 of 101 bonds at chi = 4096), "
                                 "one timed layer, no separate warm-up (the preparation columns are the warm-up)")
            if not args.no_cpu_baseline:
                rate, secs, cores = oracle_sample(wi, og)
                entry["cpu_baseline_gates_per_s"] = rate
                entry["cpu_baseline_sample"] = f"{og} synthetic saturated-bond gates, {secs:.1f} s on {cores} cores"
            per_workload[wi.name] = entry

    traffic = svd_traffic_bytes(w.name)
    out = {
        "metric": "two-site U(1) gate updates/sec", "value": value, "unit": "gates/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "c128", "data": "synthetic",
        "config": {"workload": w.name, "M": w.M, "d": w.d, "N": w.N, "chi": w.chi, "cutoff": w.cutoff,
                   "step": f"one brick-wall layer ({gates_per_step} gates, 2 launches of every kernel) on the state after "
                           f"{res['n_prep']} columns of the config's trajectory",
                   "l2": "state touched per step exceeds L2 (inputs larger than L2, no flush)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "bond_dim_max": work["bond_dim_max"], "bond_dim_median": work["bond_dim_median"],
                   "sectors_max": work["sectors_max"], "svd_blocks_per_step": work["svd_blocks"],
                   "max_block": work["max_block"]},
        "e2e": {"value": e2e, "unit": "gates/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": ms_e2e / args.steps},
        "gpu_launches": int(res["launches"]),
        "clocks": res["clocks"],
        "roofline": {"kernel": "svd_kernel (a3)", "bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                     "frac": frac, "traffic": traffic,
                     "peak_source": "derived: 148 SMs x 64 FP64 FMA/clk x 2 x sm_max_mhz (no FP64 entry in MEASURED_PEAKS.json); "
                                    "measured in this run by paper_2303_11409_b200/csrc/fp64_probe.cu: see peak_probe",
                     "peak_probe": probe,
                     "traffic_source": (f"profiles/svd_traffic_{w.name}.csv (ncu --set full, one launch of this workload)"
                                        if traffic is not None else "no committed ncu capture of this workload"),
                     "flops": "useful SVD flops 4*min(14mn^2+8n^3, 6mn^2+20n^3) per block (SURVEY §8(d))",
                     "ms_per_launch": ms_launch, "launches": svd_n,
                     "share_of_step": svd_ms / ms if ms > 0 else None},
        "useful_gflops": useful_flops_step * args.steps * world / (ms * 1e-3) / 1e9,
        "memory_bound_stages": mem or None,
        "a2_contract": {"useful_tflops": (0.5 * (work["a2_flops"] + work_after["a2_flops"]) * args.steps
                                          / (prof["a2_contract"][0] * 1e-3) / 1e12) if prof["a2_contract"][0] > 0 else None,
                        "note": "minimum-form flops 8 nL nC nR per (c_l, c', c_r) triple / summed CUDA-event time of contract_kernel"},
        "useful_frac_of_fp64_peak": useful_flops_step * args.steps * world / (ms * 1e-3) / 1e12 / (peak * world),
        "stage_ms_per_step": stage_ms,
        "trajectory": {"gates": res["prep_gates"], "ms": res["prep_ms"],
                       "gates_per_s": res["prep_gates"] / (res["prep_ms"] * 1e-3) if res["prep_ms"] > 0 else None},
        "state": {"sum_n": res["sum_n"], "log_norm": res["log_norm"], "discarded": stats["discarded"], "svd_sweeps_max": stats["sweeps"],
                  "svd_converged": stats["converged"], "full_environment_readout": res["full"], "fock_sampling": res["fock"]},
        "cpu_baseline": cpu,
        "per_workload": per_workload,
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
    ap.add_argument("--no-per-workload", action="store_true", help="skip the shorter measurements of the other four configs")
    args = ap.parse_args()
    w = inputs.WORKLOADS[args.workload]
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()

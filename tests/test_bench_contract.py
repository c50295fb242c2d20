"""CPU-side checks of bench.py's contract: the reference arm (the oracle timed on host cores) prints one valid JSON
line, under torchrun only rank 0 prints it, and the max-over-ranks helper of the N > 1 path works over gloo with
world size 2.  (The GPU arm itself needs a B200 and is exercised by the driver.)"""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
REF_ARGS = ["--impl", "reference", "--workload", "2", "--steps", "1", "--warmup", "1", "--ref-gates", "1"]
KEYS = {"impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
        "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"}


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def json_lines(text):
    return [json.loads(l) for l in text.splitlines() if l.startswith("{")]


def test_reference_arm_single_process():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + REF_ARGS, capture_output=True, text=True,
                       timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr
    lines = json_lines(r.stdout)
    assert len(lines) == 1
    d = lines[0]
    assert KEYS <= set(d)
    assert d["impl"] == "reference" and d["unit"] == "gates/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["config"]["workload"] == "hcb-M64-chi256"


def torchrun(script_args):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port())] + script_args
    return subprocess.run(cmd, capture_output=True, text=True, timeout=900, cwd=ROOT)


def test_reference_arm_two_ranks_only_rank0_prints():
    r = torchrun([os.path.join(ROOT, "bench.py"), "--gpus", "2"] + REF_ARGS)
    assert r.returncode == 0, r.stderr
    lines = json_lines(r.stdout)
    assert len(lines) == 1 and lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2


def test_max_over_ranks_gloo_world2():
    r = torchrun([os.path.join(ROOT, "tests", "_dist_max_helper.py")])
    assert r.returncode == 0, r.stderr
    out = r.stdout + r.stderr
    assert "RANK0 [2.0, 10.0]" in out and "RANK1 [2.0, 10.0]" in out, out

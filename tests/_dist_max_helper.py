"""Helper of tests/test_bench_contract.py: run under torchrun with 2 ranks on CPU (gloo)."""
import os
import sys

import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402

if __name__ == "__main__":
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    out = bench.dist_max([rank + 1.0, 10.0 - rank], world, "cpu")
    dist.barrier()
    print(f"RANK{rank} {out}")
    dist.destroy_process_group()

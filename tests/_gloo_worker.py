"""Worker of tests/test_multi_rank_cpu.py: the N > 1 host logic of bench.py under gloo (no GPU)."""
import json
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402
from paper_1702_02256_b200 import inputs  # noqa: E402


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    # (1) weak-scaling shards: every rank builds its own full-size bank from its own seed stream
    w = bench.make_workload(0, rank)
    digest = float(np.abs(w.banks[0].a1).sum())
    all_d = [None] * world
    dist.all_gather_object(all_d, digest)
    # (2) strong-style contiguous template ranges cover [0, T) exactly once
    lo, hi = inputs.shard_templates(1024, world, rank)
    ranges = [None] * world
    dist.all_gather_object(ranges, (lo, hi))
    # (3) timing rule: everyone reports the slowest rank
    slow = bench.max_over_ranks(10.0 + rank, world)
    # (4) whole-job value = units of all ranks / max time
    upd = torch.tensor([float(w.updates_per_block())], dtype=torch.float64)
    dist.all_reduce(upd)
    if rank == 0:
        print(json.dumps({"digests": all_d, "ranges": ranges, "slow": slow, "total_updates": upd.item(),
                          "per_rank_updates": w.updates_per_block(), "world": world}))
    dist.barrier()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()

"""Worker of tests/test_sharding_gloo.py: one rank of a world_size-N `gloo` group on CPU.

Exercises the host-side multi-process logic bench.py uses at N > 1 (unit sharding, max-over-ranks timing,
summary gather) without a GPU.  Prints one JSON line on rank 0."""
import json
import os
import sys

import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2301_04259_b200 import sharding  # noqa: E402


def main():
    n_units = int(sys.argv[1])
    dist.init_process_group("gloo")
    rank, world = sharding.world_info()
    b, e = sharding.shard_range(n_units, rank, world)
    mine = sharding.shard_list(list(range(n_units)), rank, world)
    assert mine == list(range(b, e))
    # per-unit summary: (unit id, unit id squared) computed by the owner only
    local = torch.tensor([[u, u * u] for u in mine], dtype=torch.float64).reshape(-1, 2)
    allrows = sharding.gather_unit_summaries(local, n_units)
    # device-timed duration stand-in: rank r reports 10 + r ms; every rank must see the max
    tmax = sharding.max_over_ranks(10.0 + rank)
    total = sharding.sum_over_ranks(float(len(mine)))
    dist.barrier()
    if rank == 0:
        print(json.dumps({"world": world, "rows": allrows.tolist(), "tmax": tmax, "total_units": total}))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()

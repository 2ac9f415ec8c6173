"""Worker of tests/test_multirank_gloo.py: one of two CPU ranks (gloo).  Checks the host-side multi-rank logic of
bench.py: per-rank workloads differ (seed offset = rank), times reduce with MAX, units with SUM."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench       # noqa: E402
import flockgen    # noqa: E402

rank, _, world = bench.dist_env()
assert world == 2
dist.init_process_group("gloo")
w = flockgen.make_config(2, seed_offset=rank, B=2)
digest = float(np.abs(w.raw.astype(np.float64)).sum())
both = [torch.zeros(1, dtype=torch.float64) for _ in range(2)]
dist.all_gather(both, torch.tensor([digest], dtype=torch.float64))
assert float(both[0]) != float(both[1]), "ranks must draw different batches"
total_ms, t_e2e, frames, cands = bench.reduce_over_ranks(10.0 + rank, 1.0 + 2 * rank, float(w.B), float(w.total_candidates), world, "cpu")
assert total_ms == 11.0 and t_e2e == 3.0, (total_ms, t_e2e)
assert frames == 4.0 and cands == 4 * 8400.0, (frames, cands)
dist.barrier()
dist.destroy_process_group()
if rank == 0:
    print("gloo worker ok")

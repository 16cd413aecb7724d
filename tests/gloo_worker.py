"""Worker of test_bench_rank_aggregation_gloo_world2 (run under torchrun, 2 CPU ranks, gloo):
bench.py's cross-rank logic -- max of the per-rank device time, sum of the points, and the
rule that only rank 0 prints the JSON line."""
import os
import sys

import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import bench  # noqa: E402

dist.init_process_group("gloo")
r, n = dist.get_rank(), dist.get_world_size()
assert n == 2
t, pts = bench.aggregate_over_ranks(10.0 + 5.0 * r, 1000 * (r + 1), device="cpu")
assert abs(t - 15.0) < 1e-12 and pts == 3000, (t, pts)
line = bench.make_line(dict(workload="test"), n_gpus=n, steps=2, warmup=1, ms_total=2 * t, points_per_step=pts)
assert line["value"] == pts / (t * 1e-3) / 1e6 and line["n_gpus"] == 2 and line["scaling"] == "weak"
assert bench.is_printing_rank() == (r == 0)
dist.barrier()
dist.destroy_process_group()
print(f"gloo_worker ok rank {r}", flush=True)

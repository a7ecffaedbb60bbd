"""Worker of tests/test_bench_cpu.py: one rank of a world_size-2 gloo job exercising bench.py's
multi-rank aggregation (replicas: barrier, max-over-ranks time, whole-job throughput)."""
import json
import os
import sys

import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import bench  # noqa: E402

rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
dist.barrier()
local = [10.0 + 5.0 * rank, 100.0 - 7.0 * rank]            # rank-dependent "timings"
got = bench.max_over_ranks(local, world)
val = bench.job_throughput(1000, 4, world, got[0])
dist.barrier()
if rank == 0:
    print(json.dumps({"max": got, "value": val}), flush=True)
dist.destroy_process_group()

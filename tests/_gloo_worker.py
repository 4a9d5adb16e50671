"""Worker for tests/test_distributed_cpu.py: world_size-2 gloo run of bench.py's multi-rank plumbing."""
import json
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from paper_2202_13532_b200 import dist_util as du   # noqa: E402

world, rank = du.init("gloo")
du.barrier()
ms_local = 10.0 + 5.0 * rank                          # rank 1 is the slow one
ms = du.max_over_ranks(ms_local)
ok = du.all_ranks_true(rank == 0)                     # false on rank 1 -> false everywhere
ok2 = du.all_ranks_true(True)
value = du.replica_throughput(1000, 3, 4, ms, world)
du.barrier()
if rank == 0:
    print(json.dumps({"world": world, "ms": ms, "ok": ok, "ok2": ok2, "value": value}), flush=True)
du.finalize()

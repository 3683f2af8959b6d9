"""Worker of tests/test_multirank.py: one rank of a world_size-2 gloo job (launched with torch.distributed.run)."""
import json
import os
import sys

import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import bench  # noqa: E402

rank = int(os.environ["RANK"])
dist.init_process_group("gloo")
dist.barrier()
# rank 0: 10 ms for 100 units, rank 1: 20 ms for 100 units  ->  job: 200 units in 20 ms
ms_max, value = bench.aggregate_replicas(10.0 * (rank + 1), 100.0, dist, "cpu")
dist.barrier()
if rank == 0:
    print(json.dumps({"ms_max": ms_max, "value": value, "world": dist.get_world_size()}))
dist.destroy_process_group()

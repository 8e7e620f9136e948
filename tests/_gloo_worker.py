"""Worker for tests/test_multirank_gloo.py (launched by torch.distributed.run, world_size 2, CPU)."""
import json
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2301_03636_b200 import replicas  # noqa: E402

g = replicas.Group(backend="gloo")
g.barrier()
my_ms = 10.0 + 5.0 * g.rank  # rank 1 is slower
mx = g.max_over_ranks(my_ms)
g.barrier()
out = {"rank": g.rank, "world": g.world, "max_ms": mx, "rate": replicas.whole_job_rate(1000.0, g.world, mx)}
with open(os.path.join(sys.argv[1], "rank%d.json" % g.rank), "w") as f:
    json.dump(out, f)
g.close()

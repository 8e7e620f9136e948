"""Worker for tests/test_multirank_gloo.py: the slab halo exchange on CPU tensors over gloo."""
import json
import os
import sys

import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2301_03636_b200 import replicas, slab  # noqa: E402

g = replicas.Group(backend="gloo")
global_dims = (4, 4, 2, 4 * g.world)  # lt = 4 slices per rank, 32 sites per slice
geom = slab.SlabGeometry(global_dims, g.world, g.rank)
nbytes = geom.slice_bytes("spinor", "f64", "soa", False)
buf = torch.zeros((geom.lt + 2) * nbytes, dtype=torch.uint8)
# interior slice k (1..lt) of rank r is filled with the byte value 10*r + k; ghosts start as 255
for k in range(geom.lt + 2):
    buf[k * nbytes:(k + 1) * nbytes] = 255 if k in (0, geom.lt + 1) else 10 * g.rank + k
reqs = slab.exchange_halos(buf, geom, nbytes, g.dist)
for r in reqs:
    r.wait()
g.barrier()
lo = buf[0:nbytes]
hi = buf[(geom.lt + 1) * nbytes:]
out = {"rank": g.rank, "world": g.world, "lo_min": int(lo.min()), "lo_max": int(lo.max()), "hi_min": int(hi.min()),
       "hi_max": int(hi.max()), "interior_ok": all(int(buf[k * nbytes]) == 10 * g.rank + k for k in range(1, geom.lt + 1)),
       "lt": geom.lt, "up": geom.up, "down": geom.down}
with open(os.path.join(sys.argv[1], "slab_rank%d.json" % g.rank), "w") as f:
    json.dump(out, f)
g.close()

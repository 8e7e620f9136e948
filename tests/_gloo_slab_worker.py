"""Worker for tests/test_multirank_gloo.py: the slab face exchange on CPU tensors over gloo."""
import json
import os
import sys

import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2301_03636_b200 import replicas, slab  # noqa: E402

g = replicas.Group(backend="gloo")
global_dims = (4, 4, 2, 4 * g.world)  # lt = 4 slices per rank, 32 sites per slice
geom = slab.SlabGeometry(global_dims, g.world, g.rank)
nbytes = geom.slice_sites * 12 * 8  # one fp64 half-spinor face
# a rank's face DOWN is filled with the byte 10 * rank + 1, its face UP with 10 * rank + 2; the receive buffers start as 255
faces = {"face_down": torch.full((nbytes,), 10 * g.rank + 1, dtype=torch.uint8),
         "face_up": torch.full((nbytes,), 10 * g.rank + 2, dtype=torch.uint8),
         "face_from_above": torch.full((nbytes,), 255, dtype=torch.uint8),
         "face_from_below": torch.full((nbytes,), 255, dtype=torch.uint8)}
for r in slab.exchange_faces(faces, geom, g.dist):
    r.wait()
g.barrier()
out = {"rank": g.rank, "world": g.world, "lt": geom.lt, "up": geom.up, "down": geom.down, "t0": geom.t0,
       "above_min": int(faces["face_from_above"].min()), "above_max": int(faces["face_from_above"].max()),
       "below_min": int(faces["face_from_below"].min()), "below_max": int(faces["face_from_below"].max()),
       "sent_intact": bool((faces["face_down"] == 10 * g.rank + 1).all() and (faces["face_up"] == 10 * g.rank + 2).all())}
with open(os.path.join(sys.argv[1], "slab_rank%d.json" % g.rank), "w") as f:
    json.dump(out, f)
g.close()

"""Multi-GPU Dslash by T-slab decomposition with half-spinor faces.

The paper runs one GPU per node and leaves multi-GPU to future work; BASELINE.json's north_star
keeps everything on one GPU, so `bench.py` defaults to independent replicas.  This module is the sharded alternative:

  * the global lattice (L_X, L_Y, L_Z, L_T) is cut along t into `world` slabs of lt = L_T / world slices; a rank's
    fields are ordinary native fields of its local lattice (L_X, L_Y, L_Z, lt): no ghost slices, links never travel;
  * per application a rank sends two FACES of spin-projected half-spinors (6 complex numbers per site of a time slice,
    half of a spinor slice): face DOWN = P^-_t in(x, 0) to the rank below, face UP = U_t^dagger P^+_t in(x, lt-1) to the
    rank above (torch.distributed P2P over NCCL / NVLink; gloo for the CPU tests).  No global collective exists;
  * the interior slices are computed while the faces fly, the two boundary slices after they have arrived.

All arithmetic and all launches sit behind the C ABI (dslash_slab_pack_faces / _interior / _boundary,
include/dslash_b200.h); this file only posts the four messages and orders the streams.
"""
import numpy as np


class SlabGeometry:
    def __init__(self, global_dims, world: int, rank: int):
        lx, ly, lz, lt = (int(d) for d in global_dims)
        if world < 1 or not (0 <= rank < world):
            raise ValueError("bad rank/world")
        if lt % world:
            raise ValueError("L_T = %d is not divisible by the number of ranks %d" % (lt, world))
        self.global_dims = (lx, ly, lz, lt)
        self.world, self.rank = world, rank
        self.lt = lt // world                      # slices per rank
        self.t0 = rank * self.lt                   # global t of local slice 0
        self.local_dims = (lx, ly, lz, self.lt)
        self.slice_sites = lx * ly * lz
        self.up = (rank + 1) % world               # owns global t0 + lt
        self.down = (rank - 1) % world


def face_messages(geom: SlabGeometry):
    """The four messages of one exchange, in the order they must be posted (the order makes world = 2, where both
    neighbours are the same peer, match correctly without tags: my first send pairs with the peer's first receive).
    Each entry: (kind, peer, buffer name)."""
    return [("send", geom.down, "face_down"),          # P^-_t in(x, 0): the forward t hop of the rank below's last slice
            ("send", geom.up, "face_up"),              # U_t^dagger P^+_t in(x, lt-1): backward t hop of the rank above's first slice
            ("recv", geom.up, "face_from_above"),      # <- the face DOWN of the rank above
            ("recv", geom.down, "face_from_below")]    # <- the face UP of the rank below


def exchange_faces(faces: dict, geom: SlabGeometry, dist=None):
    """Start the exchange of the four face buffers (flat uint8 tensors).  Returns the requests to wait on (empty when
    world == 1: the periodic wrap is two local copies).  `dist` is torch.distributed (initialised) or None."""
    if geom.world == 1:
        faces["face_from_above"].copy_(faces["face_down"])
        faces["face_from_below"].copy_(faces["face_up"])
        return []
    ops = []
    for kind, peer, name in face_messages(geom):
        fn = dist.isend if kind == "send" else dist.irecv
        ops.append(dist.P2POp(fn, faces[name], peer))
    return dist.batch_isend_irecv(ops)


def exchange_faces_in_process(all_faces, geoms):
    """The same data movement for `world` slabs that live in ONE process (single-GPU emulation of the ranks: the
    profiling guide forbids running mutually waiting ranks as separate kernels/processes on one GPU)."""
    for r, g in enumerate(geoms):
        all_faces[g.down]["face_from_above"].copy_(all_faces[r]["face_down"])
        all_faces[g.up]["face_from_below"].copy_(all_faces[r]["face_up"])


class SlabDslash:
    """One rank's share of a T-slab decomposed Dslash.  `exchange` is a callable(faces) -> requests; the default uses
    torch.distributed through `group` (a replicas.Group)."""

    def __init__(self, global_dims, precision="f64", layout="soa", recon12=False, group=None, rank=None, world=None,
                 device="cuda:0", exchange=None):
        import torch
        from . import binding as B
        from .device import Lattice
        self.torch, self.B = torch, B
        if group is not None:
            rank, world = group.rank, group.world
        self.geom = SlabGeometry(global_dims, world if world is not None else 1, rank if rank is not None else 0)
        self.group = group
        self.lat = Lattice(self.geom.local_dims, precision, layout, recon12, device=device)
        self.face_bytes = B.dslash_slab_face_bytes(self.lat.ctx)
        self.faces = {name: torch.empty(self.face_bytes, dtype=torch.uint8, device=self.lat.device)
                      for name in ("face_down", "face_up", "face_from_above", "face_from_below")}
        self._exchange = exchange
        self.comm_stream = torch.cuda.Stream(device=self.lat.device)

    def close(self):
        self.lat.close()

    @property
    def halo_bytes_per_application(self):
        """Bytes this rank SENDS per application (it receives as many)."""
        return 2 * self.face_bytes

    # -- data placement (canonical NumPy, global arrays indexed [T, Z, Y, X, ...])
    def _local(self, global_field):
        g = self.geom
        return np.ascontiguousarray(global_field[g.t0:g.t0 + g.lt])

    def upload_gauge(self, global_gauge):
        return self.lat.upload_gauge(self._local(global_gauge))

    def upload_spinor(self, global_spinor):
        return self.lat.upload_spinor(self._local(global_spinor))

    def download(self, native):
        """Canonical NumPy of the rank's slices, shape [lt, Z, Y, X, 4, 3, 2]."""
        return self.lat.download_spinor(native)

    # -- the operator
    def start_exchange(self):
        if self._exchange is not None:
            return self._exchange(self.faces)
        dist = self.group.dist if self.group is not None else None
        return exchange_faces(self.faces, self.geom, dist)

    def apply(self, out, inp, gauge):
        """out = (D in) restricted to this rank's slices."""
        torch, B, f = self.torch, self.B, self.faces
        main = torch.cuda.current_stream()
        st = main.cuda_stream
        B.dslash_slab_pack_faces(self.lat.ctx, f["face_down"].data_ptr(), f["face_up"].data_ptr(), inp.data_ptr(), gauge.data_ptr(), st)
        self.comm_stream.wait_stream(main)  # the faces are written on the main stream
        with torch.cuda.stream(self.comm_stream):
            reqs = self.start_exchange()
        B.dslash_slab_interior(self.lat.ctx, out.data_ptr(), inp.data_ptr(), gauge.data_ptr(), st)  # while the faces fly
        for r in reqs:
            r.wait()
        main.wait_stream(self.comm_stream)
        B.dslash_slab_boundary(self.lat.ctx, out.data_ptr(), inp.data_ptr(), gauge.data_ptr(), f["face_from_below"].data_ptr(),
                               f["face_from_above"].data_ptr(), st)

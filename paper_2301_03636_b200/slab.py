"""Multi-GPU Dslash by T-slab decomposition with a one-slice halo exchange.

The paper runs one GPU per node and leaves multi-GPU to future work; BASELINE.json's north_star
keeps everything on one GPU, so `bench.py` defaults to independent replicas.  This module is the sharded alternative:

  * the global lattice (L_X, L_Y, L_Z, L_T) is cut along t into `world` slabs of lt = L_T / world slices;
  * a rank's local lattice has lt + 2 slices: ghost slice 0 (global t0 - 1), interior slices 1..lt, ghost slice lt + 1;
    in every native layout a time slice is one contiguous byte range (blocked SoA: L_X*L_Y*L_Z must be a multiple of 32),
    so the exchange moves plain sub-buffers -- no pack kernels;
  * links are static: their ghost slices are filled once (only U_t of ghost slice 0 is ever read);
  * per application each rank sends its first interior spinor slice down and its last interior slice up
    (torch.distributed P2P over NCCL / NVLink; gloo for the CPU tests), computes the interior slices 2..lt-1 with
    dslash_set_time_range while the messages fly, then the two boundary slices.  No global collective exists.

Everything numerical is done by libdslash_b200.so; this file only moves bytes and sequences launches.
"""
import numpy as np

from . import replicas


class SlabGeometry:
    def __init__(self, global_dims, world: int, rank: int):
        lx, ly, lz, lt = (int(d) for d in global_dims)
        if world < 1 or not (0 <= rank < world):
            raise ValueError("bad rank/world")
        if lt % world:
            raise ValueError("L_T = %d is not divisible by the number of ranks %d" % (lt, world))
        self.global_dims = (lx, ly, lz, lt)
        self.world, self.rank = world, rank
        self.lt = lt // world                      # interior slices per rank
        self.t0 = rank * self.lt                   # global t of local interior slice 1
        self.local_dims = (lx, ly, lz, self.lt + 2)
        self.slice_sites = lx * ly * lz
        self.up = (rank + 1) % world               # owns global t + lt
        self.down = (rank - 1) % world

    def slice_bytes(self, field: str, precision: str, layout: str, recon12: bool) -> int:
        """Bytes of one time slice of a native field ("spinor" or "gauge")."""
        rb = 8 if precision == "f64" else 4
        if layout == "soa" and self.slice_sites % 32:
            raise ValueError("blocked SoA slabs need L_X*L_Y*L_Z to be a multiple of 32 (got %d)" % self.slice_sites)
        reals = 24 if field == "spinor" else 4 * (12 if recon12 else 18)
        return self.slice_sites * reals * rb


def halo_messages(geom: SlabGeometry):
    """The four messages of one exchange, in the order they must be posted (the order makes world = 2, where both
    neighbours are the same peer, match correctly without tags: my first send pairs with the peer's first receive).
    Each entry: (kind, peer, local_slice_index)."""
    return [("send", geom.down, 1),              # my first interior slice is the upper ghost of the rank below
            ("send", geom.up, geom.lt),          # my last interior slice is the lower ghost of the rank above
            ("recv", geom.up, geom.lt + 1),      # upper ghost  <- first interior slice of the rank above
            ("recv", geom.down, 0)]              # lower ghost  <- last interior slice of the rank below


def _slice_view(buf, index: int, nbytes: int):
    return buf[index * nbytes:(index + 1) * nbytes]


def exchange_halos(buf, geom: SlabGeometry, nbytes: int, dist=None):
    """Start the halo exchange of a native field held in the flat uint8 tensor `buf` (lt + 2 slices of `nbytes`).
    Returns a list of requests to wait on (empty when world == 1: the periodic wrap is two local copies).
    `dist` is torch.distributed (already initialised) or None for world == 1."""
    if geom.world == 1:
        _slice_view(buf, geom.lt + 1, nbytes).copy_(_slice_view(buf, 1, nbytes))
        _slice_view(buf, 0, nbytes).copy_(_slice_view(buf, geom.lt, nbytes))
        return []
    ops = []
    for kind, peer, idx in halo_messages(geom):
        fn = dist.isend if kind == "send" else dist.irecv
        ops.append(dist.P2POp(fn, _slice_view(buf, idx, nbytes), peer))
    return dist.batch_isend_irecv(ops)


def exchange_halos_in_process(bufs, geoms, nbytes: int):
    """The same data movement for `world` slabs that live in ONE process (single-GPU emulation of the ranks: the
    profiling guide forbids running mutually waiting ranks as separate kernels/processes on one GPU)."""
    world = len(bufs)
    for r in range(world):
        g = geoms[r]
        _slice_view(bufs[g.down], geoms[g.down].lt + 1, nbytes).copy_(_slice_view(bufs[r], 1, nbytes))
        _slice_view(bufs[g.up], 0, nbytes).copy_(_slice_view(bufs[r], g.lt, nbytes))


class SlabDslash:
    """One rank's share of a T-slab decomposed Dslash.  `exchange` is a callable(buf, nbytes) -> requests; the default
    uses torch.distributed through `group` (a replicas.Group)."""

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
        self.precision, self.layout, self.recon12 = precision, layout, recon12
        self.lat = Lattice(self.geom.local_dims, precision, layout, recon12, device=device)
        self.spinor_slice = self.geom.slice_bytes("spinor", precision, layout, recon12)
        self.gauge_slice = self.geom.slice_bytes("gauge", precision, layout, recon12)
        self._exchange = exchange
        self.comm_stream = torch.cuda.Stream(device=self.lat.device)

    def close(self):
        self.lat.close()

    # -- data placement (canonical NumPy, global arrays indexed [T, Z, Y, X, ...])
    def _local_with_ghosts(self, global_field):
        g = self.geom
        lt_glob = g.global_dims[3]
        idx = [(g.t0 - 1 + k) % lt_glob for k in range(g.lt + 2)]
        return np.ascontiguousarray(global_field[idx])

    def upload_gauge(self, global_gauge):
        """Local native links incl. both ghost slices (links are static: filled once, here straight from the global
        array every rank can generate from the seed)."""
        return self.lat.upload_gauge(self._local_with_ghosts(global_gauge))

    def upload_spinor(self, global_spinor):
        """Local native spinor; the ghost slices are deliberately zeroed -- apply() must fetch them."""
        loc = self._local_with_ghosts(global_spinor)
        loc[0] = 0
        loc[-1] = 0
        return self.lat.upload_spinor(loc)

    def download_interior(self, native):
        """Canonical NumPy of the interior slices, shape [lt, Z, Y, X, 4, 3, 2]."""
        return self.lat.download_spinor(native)[1:self.geom.lt + 1]

    # -- the operator
    def start_exchange(self, spinor):
        if self._exchange is not None:
            return self._exchange(spinor, self.spinor_slice)
        dist = self.group.dist if self.group is not None else None
        return exchange_halos(spinor, self.geom, self.spinor_slice, dist)

    def apply(self, out, inp, gauge):
        """out(interior) = D in: exchange the two boundary slices of `inp`, overlap with the interior slices."""
        torch, B, g = self.torch, self.B, self.geom
        main = torch.cuda.current_stream()
        self.comm_stream.wait_stream(main)  # `inp` was produced on the main stream
        with torch.cuda.stream(self.comm_stream):
            reqs = self.start_exchange(inp)
        if g.lt > 2:  # slices 2..lt-1 need no ghost data
            B.dslash_set_time_range(self.lat.ctx, 2, g.lt)
            self.lat.apply(out, inp, gauge)
        for r in reqs:
            r.wait()
        main.wait_stream(self.comm_stream)
        if g.lt >= 2:
            B.dslash_set_time_range(self.lat.ctx, 1, 2)
            self.lat.apply(out, inp, gauge)
            B.dslash_set_time_range(self.lat.ctx, g.lt, g.lt + 1)
            self.lat.apply(out, inp, gauge)
        else:  # a single interior slice touches both ghosts
            B.dslash_set_time_range(self.lat.ctx, 1, 2)
            self.lat.apply(out, inp, gauge)
        B.dslash_set_time_range(self.lat.ctx, 0, g.lt + 2)

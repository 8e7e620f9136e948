"""Host logic of DSLASH_KERNEL_GMARCH (no GPU): the block plan dslash_gmarch_plan() builds -- the same function whose
output dslash_set_kernel uploads -- resolves, for EVERY lane of every warp, each of the six in-slice neighbours of Eq. 1
(delta_{x+-mu^,y} on a periodic lattice) to the right source vector AND, with the kernel's lane rule, to the
right lane; covers every (vector, time slice) exactly once; pairs exchange-buffer writers and readers; counts the readers the
mbarriers are initialised with; marks exactly one "last read" per (warp, ring row); and fits the shared memory of a block."""
import collections

import pytest

FP64, FP32 = 0, 1


@pytest.fixture(scope="module")
def B():
    from paper_2301_03636_b200 import build
    build.build()
    from paper_2301_03636_b200 import binding
    return binding


def kernel_lane(lx, vec, lane, d, sign):
    """The lane rule of dslash_gmarch_kernel (csrc/dslash_gmarch.cu), restated."""
    x = (vec * 32 + lane) % lx
    if d == 0:
        if sign > 0:
            return (lane - (lx - 1)) % 32 if x + 1 == lx else (lane + 1) % 32
        return (lane + lx - 1) % 32 if x == 0 else (lane - 1) % 32
    if d == 1:
        return (lane + sign * lx) % 32
    return lane


def check_plan(B, dims, precision, recon, t0, t1, wave):
    lx, ly, lz, lt = dims
    plane = lx * ly
    shape, blocks = B.dslash_gmarch_plan(dims, precision, recon, t0, t1, wave)
    assert shape["smem_bytes"] <= 232448 and shape["nblocks"] == len(blocks) == shape["S"] * shape["G"]
    assert 1 <= shape["NW"] <= (8 if precision == FP64 else 12) and shape["NW"] == shape["units_per_block"] * shape["vecs_per_unit"]
    assert shape["NWB"] <= B.GM_NWB_MAX and shape["NLS"] >= 2 and shape["NHS"] >= 1
    cover = collections.Counter()
    halo_stages = own_vectors = 0
    for blk in blocks:
        assert t0 <= blk["t0"] and blk["nt"] >= 1 and blk["t0"] + blk["nt"] <= t1
        ws = blk["warps"]
        nact = blk["nact"]
        assert 1 <= nact <= shape["NW"] and all(w["vec"] >= 0 for w in ws[:nact]) and all(w["vec"] < 0 for w in ws[nact:])
        local = {w["vec"]: i for i, w in enumerate(ws[:nact])}
        assert len(local) == nact
        ring_readers = collections.Counter()
        wbuf_readers = collections.Counter()
        wbuf_owner = {}
        for i, w in enumerate(ws[:nact]):
            for d in range(3):
                if w["wr"][d] >= 0:
                    assert 0 <= w["wr"][d] < shape["NWB"] and w["wr"][d] not in wbuf_owner
                    wbuf_owner[w["wr"][d]] = (i, d)
        for i, w in enumerate(ws[:nact]):
            v = w["vec"]
            shared = 0
            for d in range(3):
                assert 1 <= len(w["f"][d]) <= B.GM_SRC_MAX and 1 <= len(w["b"][d]) <= B.GM_SRC_MAX
                for entries in (w["f"][d], w["b"][d]):
                    masks = [m for (_, m) in entries]
                    assert all(m for m in masks) and sum(masks) == 0xFFFFFFFF  # disjoint, every lane served exactly once
                    acc = 0
                    for m in masks:
                        assert acc & m == 0
                        acc |= m
            for lane in range(32):
                s = v * 32 + lane
                x, y, z = s % lx, (s // lx) % ly, s // plane
                assert z < lz
                nf = (s - x + (x + 1) % lx, s + ((y + 1) % ly - y) * lx, s + ((z + 1) % lz - z) * plane)
                nb = (s - x + (x - 1) % lx, s + ((y - 1) % ly - y) * lx, s + ((z - 1) % lz - z) * plane)
                for d in range(3):
                    (fid, _), = [(e, m) for (e, m) in w["f"][d] if (m >> lane) & 1]
                    src = ws[fid & 0xFF]["vec"] if fid >= 0 else -fid - 1
                    assert src == nf[d] // 32 and kernel_lane(lx, v, lane, d, +1) == nf[d] % 32
                    assert (fid >= 0) == (nf[d] // 32 in local)  # a vector of the block is served from the ring
                    if fid < 0:
                        shared |= 1 << d
                    (bid, _), = [(e, m) for (e, m) in w["b"][d] if (m >> lane) & 1]
                    if bid >= 0:
                        owner, od = wbuf_owner[bid]
                        src = ws[owner]["vec"]
                        assert od == d
                    else:
                        src = -bid - 1
                        assert d != 0  # x neighbours never leave the block
                    assert src == nb[d] // 32 and kernel_lane(lx, v, lane, d, -1) == nb[d] % 32
            assert w["link_shared"] == shared and not shared & 1
            # ring rows: one "last read" per row this warp reads as a forward source, and it is the last one in program order
            reads = [(d, e, fid) for d in range(3) for e, (fid, _) in enumerate(w["f"][d]) if fid >= 0]
            rows = {fid & 0xFF for (_, _, fid) in reads}
            for r in rows:
                mine = [(d, e, fid) for (d, e, fid) in reads if fid & 0xFF == r]
                assert [bool(fid & 0x100) for (_, _, fid) in mine] == [False] * (len(mine) - 1) + [True]
                ring_readers[r] += 1
            assert w["own_done"] == (0 if i in rows else 1)
            if i not in rows:
                ring_readers[i] += 1
            for d in range(3):
                for (bid, _) in w["b"][d]:
                    if bid >= 0:
                        wbuf_readers[bid] += 1
            nh = sum(1 for d in (1, 2) for (fid, _) in w["f"][d] if fid < 0) + sum(1 for d in (1, 2) for (bid, _) in w["b"][d] if bid < 0)
            nl = 4 + sum(1 for d in (1, 2) for (bid, _) in w["b"][d] if bid < 0)
            assert nh <= 12 and nl <= 12  # the producers' stage tables
            halo_stages += (nh + nl - 4) * blk["nt"]
            own_vectors += blk["nt"]
            for t in range(blk["t0"], blk["t0"] + blk["nt"]):
                cover[(v, t)] += 1
        assert [blk["ring_readers"][r] for r in range(nact)] == [ring_readers[r] for r in range(nact)]
        assert set(wbuf_readers) == set(wbuf_owner)  # a buffer is written only if somebody reads it
        assert all(blk["wbuf_readers"][b] == n for b, n in wbuf_readers.items())
    assert len(cover) == (lx * ly * lz // 32) * (t1 - t0) and set(cover.values()) == {1}
    return shape, halo_stages / own_vectors


@pytest.mark.parametrize("dims,precision,recon", [
    ((48, 48, 48, 96), FP32, 18),   # BASELINE.json configs[3]: a vector is 2/3 of an x row
    ((48, 48, 48, 96), FP32, 12),
    ((24, 24, 24, 24), FP64, 18),   # configs[4]: 4/3 of a row
    ((16, 16, 16, 16), FP64, 18),   # configs[1]: two rows per vector
    ((32, 32, 32, 64), FP64, 18),   # the L_X == 32 case the specialised kernel covers
    ((32, 16, 12, 9), FP32, 12),
    ((64, 16, 16, 16), FP32, 18),   # two vectors per row
    ((8, 8, 8, 8), FP64, 12),       # four rows per vector: y neighbours inside the vector
    ((40, 8, 4, 4), FP32, 18),      # lcm(40, 32) = 160: five vectors per unit
    ((16, 4, 2, 4), FP64, 18),
    ((4, 8, 1, 3), FP64, 18),       # L_Z = 1: a vector is its own z neighbour
    ((2, 16, 3, 2), FP32, 18),
    ((96, 2, 2, 2), FP32, 18),
])
def test_plan_resolves_every_neighbour(B, dims, precision, recon):
    check_plan(B, dims, precision, recon, 0, dims[3], 148)


def test_time_range_and_small_waves(B):
    check_plan(B, (48, 48, 48, 96), FP32, 18, 5, 37, 148)
    check_plan(B, (24, 24, 24, 24), FP64, 18, 23, 24, 148)
    check_plan(B, (16, 16, 16, 16), FP64, 18, 0, 16, 4)
    check_plan(B, (48, 8, 8, 8), FP32, 18, 0, 8, 1)


def test_config4_decomposition_is_what_design_md_says(B):
    # 48^3 x 96 fp32: units of 96 sites (2 rows, 3 vectors), 4 units = 12 compute warps per block, two full waves of 148 blocks
    shape, halo = check_plan(B, (48, 48, 48, 96), FP32, 18, 0, 96, 148)
    assert (shape["vecs_per_unit"], shape["units_per_block"], shape["NW"], shape["G"]) == (3, 4, 12, 1)
    assert shape["nblocks"] == 296
    # halo stages (spinor or link vectors fetched a second time) per own vector and step: 30 distinct vectors around a 2 x 2
    # patch of units (2.5), more because a half-used vector is fetched by each of the two warps that need it
    assert halo < 3.6


def test_ineligible_lattices_are_refused(B):
    for dims in ((48, 3, 4, 4), (33, 32, 4, 4), (12, 2, 2, 2)):  # L_X * L_Y not a multiple of 32, or a unit of too many vectors
        with pytest.raises(Exception):
            B.dslash_gmarch_plan(dims, FP32, 18, 0, dims[3], 148)
    with pytest.raises(Exception):
        B.dslash_gmarch_plan((48, 48, 48, 96), FP32, 18, 3, 3, 148)


def test_seeded_random_geometries(B):
    """Forty seeded random lattices (every x extent from 1 to 96 that the kernel accepts has a chance): whatever the unit shape,
    the plan resolves every neighbour.  Lattices the library refuses must be exactly the ineligible ones."""
    import math
    import random
    rnd = random.Random(230103636)
    checked = 0
    while checked < 40:
        lx = rnd.choice([1, 2, 3, 4, 6, 8, 12, 16, 20, 24, 32, 40, 48, 64, 80, 96])
        ly, lz, lt = rnd.randint(1, 12), rnd.randint(1, 5), rnd.randint(1, 5)
        precision, recon = rnd.choice([FP64, FP32]), rnd.choice([18, 12])
        unit_vectors = lx // math.gcd(lx, 32)  # lcm(L_X, 32) / 32
        eligible = (lx * ly) % 32 == 0 and unit_vectors <= (8 if precision == FP64 else 12)
        try:
            check_plan(B, (lx, ly, lz, lt), precision, recon, 0, lt, rnd.choice([1, 7, 148]))
            assert eligible, (lx, ly, lz, lt)
            checked += 1
        except B.DslashError:
            # refused: ineligible, or eligible in principle but no decomposition fits the shared memory of a block
            assert not eligible or (precision == FP64 and unit_vectors >= 5), (lx, ly, lz, lt, precision)

"""Host logic of DSLASH_KERNEL_MARCH (no GPU): the block plan dslash_march_plan() builds -- the same function whose
output dslash_set_kernel uploads -- covers every (row, time slice) exactly once, describes the neighbour relations of
Eq. 1's periodic (y,z) plane correctly (delta_{x+-mu^,y} on a periodic lattice), pairs every exchange-buffer
writer with exactly one reader, and keeps the halo small enough for the traffic the design claims."""
import collections

import pytest


@pytest.fixture(scope="module")
def B():
    from paper_2301_03636_b200 import build
    build.build()
    from paper_2301_03636_b200 import binding
    return binding


def check_plan(B, dims, t0, t1, wave):
    lx, ly, lz, lt = dims
    blocks = B.dslash_march_plan(dims, t0, t1, wave)
    cover = collections.Counter()
    halo_f = halo_b = rows = 0
    for blk in blocks:
        assert t0 <= blk["t0"] and blk["nt"] >= 1 and blk["t0"] + blk["nt"] <= t1
        ws = blk["warps"]
        act = [w for w in ws if w["row"] >= 0]
        assert len(act) == blk["nact"] >= 1
        assert all(w["row"] >= 0 for w in ws[:blk["nact"]])  # active warps first
        local = {w["row"]: i for i, w in enumerate(ws) if w["row"] >= 0}
        assert len(local) == len(act)
        writers, readers = {}, {}
        for i, w in enumerate(act):
            y, z = w["row"] % ly, w["row"] // ly
            assert 0 <= z < lz
            nf = ((y + 1) % ly + ly * z, y + ly * ((z + 1) % lz))
            nb = ((y - 1) % ly + ly * z, y + ly * ((z - 1) % lz))
            for d in range(2):
                assert w["bwd"][d] == nb[d]
                if w["fwd"][d] >= 0:
                    assert ws[w["fwd"][d]]["row"] == nf[d]
                else:
                    assert -w["fwd"][d] - 1 == nf[d] and nf[d] not in local
                    halo_f += blk["nt"]
                if w["wr"][d] >= 0:
                    assert w["fwd"][d] >= 0 and (d, w["wr"][d]) not in writers and 0 <= w["wr"][d] < B.MARCH_NWS
                    writers[(d, w["wr"][d])] = w["fwd"][d]  # consumer warp
                if w["rd"][d] >= 0:
                    assert nb[d] in local and (d, w["rd"][d]) not in readers
                    readers[(d, w["rd"][d])] = i
                else:
                    halo_b += blk["nt"]
                # the neighbour is a row of this block  <=>  it is served from shared memory (no slot shortage here)
                assert (nb[d] in local) == (w["rd"][d] >= 0)
            for t in range(blk["t0"], blk["t0"] + blk["nt"]):
                cover[(w["row"], t)] += 1
            rows += blk["nt"]
        assert writers == readers  # every buffer: one writer, one reader, and the reader is the writer's forward neighbour
        slots = [s for (_, s) in writers]
        assert len(slots) == len(set(slots))  # buffers are not shared between directions either
    assert len(cover) == ly * lz * (t1 - t0) and set(cover.values()) == {1}
    return blocks, halo_f / rows, halo_b / rows


def test_bench_lattice_is_one_wave_of_7_and_6_row_patches(B):
    dims = (32, 32, 32, 64)
    blocks, hf, hb = check_plan(B, dims, 0, 64, 148)
    assert len(blocks) == 148 and all(b["t0"] == 0 and b["nt"] == 64 for b in blocks)
    assert sorted(set(b["nact"] for b in blocks)) == [6, 7]
    # L2 -> SM bytes per site (fp64, 18-real): own spinor 192 + own links 576 + forward halo spinors 192 each + backward halo
    # spinor and link 336 each; the design quotes 1.23 KB
    per_site = 192 + 576 + 192 * hf + 336 * hb
    assert per_site <= 1250, per_site


@pytest.mark.parametrize("dims,t0,t1,wave", [
    ((32, 4, 4, 8), 0, 8, 148), ((32, 4, 4, 8), 1, 7, 148), ((32, 1, 1, 1), 0, 1, 148), ((32, 2, 1, 3), 0, 3, 148),
    ((32, 5, 3, 2), 0, 2, 148), ((32, 16, 12, 9), 0, 9, 148), ((32, 40, 30, 3), 0, 3, 148), ((32, 32, 32, 64), 16, 48, 148),
    ((32, 32, 32, 64), 0, 64, 132), ((32, 32, 32, 64), 0, 64, 1), ((32, 7, 9, 5), 2, 5, 8), ((32, 48, 48, 96), 0, 96, 148),
])
def test_plans_cover_every_row_and_slice_once(B, dims, t0, t1, wave):
    check_plan(B, dims, t0, t1, wave)


def test_plan_argument_errors(B):
    for dims, t0, t1, wave in [((16, 4, 4, 4), 0, 4, 148), ((32, 4, 4, 4), 2, 2, 148), ((32, 4, 4, 4), 0, 5, 148),
                               ((32, 4, 4, 4), 0, 4, 0)]:
        with pytest.raises(B.DslashError) as e:
            B.dslash_march_plan(dims, t0, t1, wave)
        assert e.value.status == B.DSLASH_ERR_UNSUPPORTED
    with pytest.raises(B.DslashError) as e:
        B.dslash_march_plan((32, 0, 4, 4), 0, 4, 148)
    assert e.value.status == B.DSLASH_ERR_DIMS

"""GPU parity: the CUDA library (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star; metric = checks.parity_error, DESIGN.md Reading R10):
    FP64 (18- and 12-real links)  e <= 1e-12
    FP32                          e <= 1e-5   (oracle fed the fp32-rounded inputs promoted to fp64)
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-5}
SEED = 230103636


@pytest.fixture(scope="module")
def env():
    import torch
    import oracle
    from paper_2301_03636_b200 import binding, checks, device, inputs
    assert torch.cuda.is_available()

    class E:
        pass
    e = E()
    e.torch, e.oracle, e.B, e.checks, e.device, e.inputs = torch, oracle, binding, checks, device, inputs
    return e


_FIELD_CACHE = {}


def fields_and_ref(env, dims, seed, precision, full=True, nsample=4096):
    key = (tuple(dims), seed, precision, full)
    if key not in _FIELD_CACHE:
        _FIELD_CACHE.clear()  # keep one lattice at a time in host memory
        g, p = env.inputs.fields(dims, seed, precision)
        g64, p64 = env.inputs.promote(g), env.inputs.promote(p)
        if full:
            sites = None
            ref = env.oracle.dslash(p64, g64, dims)
        else:
            sites = env.inputs.sample_sites(dims, nsample, seed)
            ref = env.oracle.dslash_sites(p64, g64, dims, sites)
        _FIELD_CACHE[key] = (g, p, ref, sites)
    return _FIELD_CACHE[key]


def gpu_vs_ref(env, lat, g, p, ref, sites=None):
    out = lat.dslash(g, p)
    if sites is not None:
        out = out.reshape(-1, 4, 3, 2)[sites]
    return env.checks.parity_error(out, ref)


ALL_MODES = [(lay, r12) for lay in ("aos", "soa") for r12 in (False, True)]


# ---------------------------------------------------------------- config 1: 4^4 FP64 (+ FP32), every layout
@pytest.mark.parametrize("precision", ["f64", "f32"])
@pytest.mark.parametrize("layout,recon12", ALL_MODES)
def test_config1_4x4x4x4(env, precision, layout, recon12):
    dims = (4, 4, 4, 4)
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 1, precision)
    with env.device.Lattice(dims, precision, layout, recon12) as lat:
        assert gpu_vs_ref(env, lat, g, p, ref) <= TOL[precision]
        n0 = env.B.dslash_launch_count(lat.ctx)
        o, pi, gi = lat.new_spinor(), lat.upload_spinor(p), lat.upload_gauge(g)
        n1 = env.B.dslash_launch_count(lat.ctx)
        lat.apply(o, pi, gi)
        assert env.B.dslash_launch_count(lat.ctx) == n1 + 1  # exactly one kernel per apply
        assert n1 >= n0


# ---------------------------------------------------------------- ragged / degenerate lattices
@pytest.mark.parametrize("dims", [(4, 6, 8, 10), (3, 5, 7, 2), (2, 2, 2, 2), (1, 1, 1, 1), (1, 2, 3, 4), (33, 3, 2, 5),
                                  (10, 4, 6, 2)])
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_ragged_and_degenerate_extents(env, dims, precision):
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 11, precision)
    for layout, recon12 in ALL_MODES:
        with env.device.Lattice(dims, precision, layout, recon12) as lat:
            assert gpu_vs_ref(env, lat, g, p, ref) <= TOL[precision], (layout, recon12, "tuned")
            for depth, tpb, spt in [(4, 64, 1), (3, 128, 2), (2, 256, 4), (1, 512, 1), (4, 1024, 4)]:
                lat.set_variant(depth, tpb, spt)
                assert gpu_vs_ref(env, lat, g, p, ref) <= TOL[precision], (layout, recon12, depth, tpb, spt)


@pytest.mark.parametrize("tile", [(32, 1, 1, 1), (8, 4, 4, 1), (4, 4, 4, 4), (2, 2, 2, 4), (16, 2, 2, 2), (8, 8, 8, 2),
                                  (1, 1, 1, 32), (16, 4, 4, 4)])
def test_tuned_kernel_every_tile_shape(env, tile):
    dims = (12, 6, 10, 5)
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 12, "f64")
    with env.device.Lattice(dims, "f64", "soa", False) as lat:
        lat.set_tile(tile)
        assert env.B.dslash_get_tile(lat.ctx) == tuple(tile)
        assert gpu_vs_ref(env, lat, g, p, ref) <= TOL["f64"]


@pytest.mark.parametrize("dims,tile,zblock", [
    ((8, 4, 12, 3), (8, 4, 2, 1), 2), ((8, 4, 12, 3), (8, 4, 2, 1), 4), ((8, 4, 12, 3), (8, 4, 2, 1), 6),
    ((8, 4, 12, 3), (8, 4, 2, 1), 12),      # one block: the plain order
    ((8, 4, 12, 3), (8, 4, 2, 1), 3),       # not a multiple of the tile's z extent: the automatic choice
    ((12, 6, 10, 5), (4, 4, 2, 1), 2), ((12, 6, 9, 4), (4, 2, 4, 2), 0),  # ragged in y and z with partial tiles
])
def test_direct_kernel_z_blocked_tile_order(env, dims, tile, zblock):
    """The block order x, y, z inside a z block, t, z block (DSLASH_OPT_PIPE_ZBLOCK) visits every site exactly once."""
    B = env.B
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 15, "f64")
    with env.device.Lattice(dims, "f64", "soa", False) as lat:
        lat.set_tile(tile)
        gi, pi, o = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
        lat.apply(o, pi, gi)
        plain = lat.download_spinor(o)
        if zblock and dims[2] % zblock == 0:
            B.dslash_set_option(lat.ctx, B.DSLASH_OPT_PIPE_ZBLOCK, zblock)
        o.fill_(0x7f)
        lat.apply(o, pi, gi)
        got = lat.download_spinor(o)
        assert env.checks.parity_error(got, ref) <= TOL["f64"]
        assert np.array_equal(got, plain)
        for op in (B.DSLASH_OP_D_DAGGER, B.DSLASH_OP_M):  # the operator kernels share the block decode
            o.fill_(0x7f)
            lat.apply_op(op, 0.3, o, pi, gi)
            assert np.isfinite(lat.download_spinor(o)).all()


# ---------------------------------------------------------------- x hops by warp shuffle (DSLASH_OPT_X_SHUFFLE)
@pytest.mark.parametrize("dims,tile", [
    ((32, 3, 5, 2), (32, 2, 2, 1)),   # one row per warp, ragged tiles in y and z (clamped rows that do not store)
    ((32, 4, 2, 3), (32, 1, 1, 2)),   # ragged in t
    ((16, 3, 3, 3), (16, 2, 2, 1)),   # two rows per warp, one of them beyond the edge in some warps
    ((8, 5, 3, 2), (8, 4, 2, 1)),     # four rows per warp
    ((4, 6, 2, 5), (4, 4, 2, 2)),
    ((2, 3, 2, 5), (2, 4, 2, 4)),     # L_X = 2: x+1 and x-1 are the same lane
    ((1, 2, 3, 4), (1, 2, 4, 4)),     # L_X = 1: the neighbour is the site itself
    ((16, 4, 4, 4), (16, 4, 4, 4)),   # 1024-thread tile
])
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_x_shuffle_kernel_matches_the_oracle_and_the_loading_kernel_bit_for_bit(env, dims, tile, precision):
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 14, precision)
    for layout, recon12 in ALL_MODES:
        with env.device.Lattice(dims, precision, layout, recon12) as lat:
            lat.set_tile(tile)
            assert env.B.dslash_get_option(lat.ctx, env.B.DSLASH_OPT_X_SHUFFLE) == (1 if precision == "f64" else 0)  # default
            gi, pi = lat.upload_gauge(g), lat.upload_spinor(p)
            outs = {}
            for on in (1, 0):
                env.B.dslash_set_option(lat.ctx, env.B.DSLASH_OPT_X_SHUFFLE, on)
                o = lat.new_spinor()
                o.fill_(0x7f)  # a site the kernel forgot to store would stay NaN-like garbage
                lat.apply(o, pi, gi)
                outs[on] = lat.download_spinor(o)
                assert env.checks.parity_error(outs[on], ref) <= TOL[precision], (layout, recon12, on)
            # same arithmetic in the same order; with 12-real links the shuffle path rebuilds row 2 of U_x(s) once for
            # both hops, from the same two rows: still the same bits
            assert np.array_equal(outs[1], outs[0]), (layout, recon12)


# ---------------------------------------------------------------- the block-cooperative marching kernel (SoA, L_X = 32)
MARCH_DIMS = [
    (32, 4, 4, 8),       # 16 rows: 1-row .. 7-row patches depending on the SM count, all wraps
    (32, 1, 1, 1),       # one row: every neighbour is the row itself (the warp exchanges with itself), t+1 == t-1 == t
    (32, 2, 1, 3),       # y+1 == y-1, z neighbour == self
    (32, 5, 3, 2),       # odd extents: a strip of one z plane, t+1 == t-1
    (32, 2, 2, 5),       # a single 4-row patch when the plan has one segment
    (32, 16, 12, 9),     # 192 rows
    (32, 32, 32, 4),     # 1024 rows: the 7/6-row patches of the bench lattice, one wave, four steps
    (32, 40, 30, 3),     # 1200 rows: more than one wave of 7-row patches on 148 SMs
]


@pytest.mark.parametrize("dims", MARCH_DIMS)
@pytest.mark.parametrize("precision", ["f64", "f32"])
@pytest.mark.parametrize("recon12", [False, True])
def test_marching_kernel_matches_the_oracle_and_the_direct_kernel_bit_for_bit(env, dims, precision, recon12):
    B = env.B
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 19, precision)
    with env.device.Lattice(dims, precision, "soa", recon12) as lat:
        gi, pi, o = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
        lat.apply(o, pi, gi)
        direct = lat.download_spinor(o)
        lat.set_kernel("march")
        assert B.dslash_get_kernel(lat.ctx) == B.DSLASH_KERNEL_MARCH
        o.fill_(0x7f)  # a site the kernel forgot to store would stay garbage
        n0 = B.dslash_launch_count(lat.ctx)
        lat.apply(o, pi, gi)
        assert B.dslash_launch_count(lat.ctx) == n0 + 1
        got = lat.download_spinor(o)
        assert env.checks.parity_error(got, ref) <= TOL[precision]
        assert np.array_equal(got, direct)  # same arithmetic, same order of the sum
        # a second application on the same context gives the same bits (no state left behind by the first)
        o.fill_(0x7f)
        lat.apply(o, pi, gi)
        assert np.array_equal(lat.download_spinor(o), direct)
        # time ranges (multi-GPU slab interior, single slices at the ends): only their slices are written
        lt = dims[3]
        for t0, t1 in [(1, lt - 1), (0, 1), (lt - 1, lt), (lt // 2, lt)]:
            if not (0 <= t0 < t1 <= lt):
                continue
            B.dslash_set_time_range(lat.ctx, t0, t1)
            o.zero_()
            lat.apply(o, pi, gi)
            part = lat.download_spinor(o)
            assert np.array_equal(part[t0:t1], direct[t0:t1]), (t0, t1)
            assert not part[:t0].any() and not part[t1:].any(), (t0, t1)


@pytest.mark.parametrize("dims", [(32, 16, 12, 9), (32, 32, 32, 4), (32, 40, 30, 3)])  # the last one: more than one wave
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_marching_kernel_options_keep_the_bits(env, dims, precision):
    """DSLASH_OPT_MARCH_POLICY changes the producers' gating (bit 16: late ring fill) and the copies' L2 hints;
    DSLASH_OPT_MARCH_LEAD > 0 adds cross-block progress counters that accumulate over launches (the plan's epoch).  Every
    combination, 20 back-to-back launches each on a non-blocking stream of ONE context (so the counters run through many
    epochs, lead-0 launches in between included -- a round-2 advisor finding: those must not move the throttle's target), has
    to give the direct kernel's bits.  A multi-wave plan switches the throttle off by itself; a new time range resets the epoch."""
    B, torch = env.B, env.torch
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 41, precision)
    with env.device.Lattice(dims, precision, "soa", False) as lat:
        gi, pi, o = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
        lat.apply(o, pi, gi)
        direct_dev = o.clone()
        assert env.checks.parity_error(lat.download_spinor(o), ref) <= TOL[precision]
        lat.set_kernel("march")
        torch.cuda.synchronize()
        st = torch.cuda.Stream()

        def run(n=20):
            o.fill_(0x7f)
            torch.cuda.synchronize()
            for _ in range(n):
                B.dslash_apply(lat.ctx, o.data_ptr(), pi.data_ptr(), gi.data_ptr(), st.cuda_stream)
            st.synchronize()
            return bool(torch.equal(o, direct_dev))

        for policy in (0, 4, 12, 16, 28, 29, -1):
            B.dslash_set_option(lat.ctx, B.DSLASH_OPT_MARCH_POLICY, policy)
            assert B.dslash_get_option(lat.ctx, B.DSLASH_OPT_MARCH_POLICY) == policy
            for lead in (0, 1, 4, 0, 2):
                B.dslash_set_option(lat.ctx, B.DSLASH_OPT_MARCH_LEAD, lead)
                assert run(), (policy, lead)
        # the direct kernel's option no longer reaches the marching kernel: 16 there means "t loads bypass L1"
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_L2_POLICY, 16)
        assert run(3) and B.dslash_get_option(lat.ctx, B.DSLASH_OPT_MARCH_POLICY) == -1
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_L2_POLICY, -1)
        # a new time range rebuilds the plan (fresh counters, epoch 0) with the throttle still on
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_MARCH_LEAD, 1)
        lt = dims[3]
        B.dslash_set_time_range(lat.ctx, 1, lt)
        o.zero_()
        torch.cuda.synchronize()
        for _ in range(5):
            B.dslash_apply(lat.ctx, o.data_ptr(), pi.data_ptr(), gi.data_ptr(), st.cuda_stream)
        st.synchronize()
        nat = B.dslash_spinor_bytes(lat.ctx) // lt  # a time slice of a blocked-SoA field with L_X = 32 is a whole number of vectors
        assert torch.equal(o[nat:], direct_dev[nat:]) and not o[:nat].any()
        B.dslash_set_time_range(lat.ctx, 0, lt)
        assert run()


def test_marching_kernel_throttle_is_not_left_behind_by_unthrottled_launches(env):
    """Round-2 advisor finding: launches with DSLASH_OPT_MARCH_LEAD = 0 used to advance the epoch the throttle's target is
    derived from, while only throttled launches advance the counters; once the option was switched on, every ring queue then
    waited out its patience (~50 us) in every launch.  Timed: throttled launches after 50 unthrottled ones must not be slower
    than throttled launches on a fresh context (best of three, 10 % margin; the defect costs 15 % and more)."""
    B, torch = env.B, env.torch
    dims = (32, 32, 32, 16)
    g, p = env.inputs.fields(dims, SEED + 43, "f64")

    def timed(lat, gi, pi, o, n=20):
        best = None
        for _ in range(3):
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(n):
                lat.apply(o, pi, gi)
            b.record()
            torch.cuda.synchronize()
            ms = a.elapsed_time(b) / n
            best = ms if best is None else min(best, ms)
        return best

    with env.device.Lattice(dims, "f64", "soa", False) as lat:
        gi, pi, o = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
        lat.apply(o, pi, gi)
        direct_dev = o.clone()
        lat.set_kernel("march")
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_MARCH_LEAD, 2)
        for _ in range(10):
            lat.apply(o, pi, gi)
        fresh = timed(lat, gi, pi, o)
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_MARCH_LEAD, 0)
        for _ in range(50):
            lat.apply(o, pi, gi)
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_MARCH_LEAD, 2)
        o.fill_(0x7f)
        after = timed(lat, gi, pi, o)
        assert torch.equal(o, direct_dev)
        assert after <= 1.10 * fresh, (fresh, after)


def test_marching_kernel_refuses_what_it_cannot_run(env):
    B = env.B
    for dims, layout in [((32, 4, 4, 4), "aos"),   # AoS rows are not contiguous vectors
                         ((16, 4, 4, 4), "soa"),   # two x rows per 32-site vector
                         ((64, 4, 4, 4), "soa")]:  # an x row is two vectors
        with env.device.Lattice(dims, "f64", layout, False) as lat:
            lat.set_kernel("march")
            o, p, g = lat.new_spinor(), lat.new_spinor(), lat.new_gauge()
            assert B.dslash_apply_status(lat.ctx, o.data_ptr(), p.data_ptr(), g.data_ptr()) == B.DSLASH_ERR_UNSUPPORTED, dims
            lat.set_kernel("auto")
            assert B.dslash_apply_status(lat.ctx, o.data_ptr(), p.data_ptr(), g.data_ptr()) == B.DSLASH_OK
            with pytest.raises(B.DslashError):
                B.dslash_set_kernel(lat.ctx, 2)  # a kernel of round 1 that no longer exists
            with pytest.raises(B.DslashError):
                B.dslash_set_kernel(lat.ctx, 7)  # the generalised marching kernel of round 2, removed in round 3


@pytest.mark.parametrize("kernel", ["march", "wpipe"])
def test_staged_kernels_on_a_non_blocking_stream_and_fresh_context(env, kernel):
    """The staged kernels keep device-side state (row counters / block plan).  A fresh context whose FIRST launch runs on a
    cudaStreamNonBlocking stream (every torch.cuda.Stream is one) must be correct: nothing may depend on the legacy default
    stream having run first (round-1 advisor finding on the counter memset)."""
    B, torch = env.B, env.torch
    dims = (32, 8, 6, 5)
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 29, "f64")
    for attempt in range(3):
        with env.device.Lattice(dims, "f64", "soa", False) as lat:
            gi, pi = lat.upload_gauge(g), lat.upload_spinor(p)
            torch.cuda.synchronize()
            st = torch.cuda.Stream()
            lat.set_kernel(kernel)
            o = lat.new_spinor()
            o.fill_(0x7f)
            torch.cuda.synchronize()
            for _ in range(4):  # back-to-back launches on the side stream
                B.dslash_apply(lat.ctx, o.data_ptr(), pi.data_ptr(), gi.data_ptr(), st.cuda_stream)
            st.synchronize()
            assert env.checks.parity_error(lat.download_spinor(o), ref) <= TOL["f64"], attempt


# ---------------------------------------------------------------- the warp-pipelined kernel (SoA, L_X = 32), selected explicitly
@pytest.mark.parametrize("dims", [
    (32, 4, 4, 8),       # several rows per warp, all wraps
    (32, 1, 1, 1),       # one row: every neighbour is the row itself
    (32, 2, 1, 3),       # y+1 == y-1, z neighbour == self
    (32, 5, 3, 2),       # odd extents, t+1 == t-1
    (32, 16, 12, 9),     # 1728 rows: more rows than resident warps on any configuration (persistent loop, tail)
])
@pytest.mark.parametrize("slots,warps,zblock", [(0, 0, 0), (2, 1, 0), (3, 2, 0), (4, 4, 0), (2, 4, 1), (3, 1, 3)])
@pytest.mark.parametrize("precision", ["f64", "f32"])
@pytest.mark.parametrize("recon12", [False, True])
def test_warp_pipelined_kernel_matches_the_oracle_and_the_direct_kernel_bit_for_bit(env, dims, slots, warps, zblock, precision, recon12):
    B = env.B
    if zblock and dims[2] % zblock:
        pytest.skip("z block does not divide L_Z")
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 23, precision)
    with env.device.Lattice(dims, precision, "soa", recon12) as lat:
        gi, pi, o = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
        lat.apply(o, pi, gi)
        direct = lat.download_spinor(o)
        lat.set_kernel("wpipe")
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_PIPE_SLOTS, slots)
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_PIPE_WARPS, warps)
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_PIPE_ZBLOCK, zblock)
        assert B.dslash_get_kernel(lat.ctx) == B.DSLASH_KERNEL_WARP_PIPE
        assert B.dslash_get_option(lat.ctx, B.DSLASH_OPT_PIPE_SLOTS) == slots
        o.zero_()
        lat.apply(o, pi, gi)
        got = lat.download_spinor(o)
        assert env.checks.parity_error(got, ref) <= TOL[precision]
        assert np.array_equal(got, direct)  # same arithmetic in the same order
        if dims[3] >= 4:  # a time range (multi-GPU slab interior): only its slices are written
            B.dslash_set_time_range(lat.ctx, 1, dims[3] - 1)
            o.zero_()
            lat.apply(o, pi, gi)
            part = lat.download_spinor(o)
            assert np.array_equal(part[1:-1], direct[1:-1]) and not part[0].any() and not part[-1].any()


def test_warp_pipelined_kernel_refill_is_ordered_after_the_reads_of_the_slot(env):
    """Regression: a slot is refilled by the ASYNC proxy right after it was read through the generic proxy; without
    fence.proxy.async 9 % of the launches of this configuration (fp32, 3 slots, 13 one-warp blocks per SM, lattice resident
    in L2 so that the bulk copies land within a few hundred cycles) returned one wrong row.  200 launches, bit for bit."""
    B, torch = env.B, env.torch
    dims = (32, 16, 12, 9)
    g, p = env.inputs.fields(dims, SEED + 25, "f32", check=False)
    with env.device.Lattice(dims, "f32", "soa", False) as lat:
        gi, pi, o1, o2 = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor(), lat.new_spinor()
        lat.apply(o1, pi, gi)
        lat.set_kernel("wpipe")
        for slots, warps in ((3, 1), (3, 2)):
            B.dslash_set_option(lat.ctx, B.DSLASH_OPT_PIPE_SLOTS, slots)
            B.dslash_set_option(lat.ctx, B.DSLASH_OPT_PIPE_WARPS, warps)
            for _ in range(100):
                o2.zero_()
                lat.apply(o2, pi, gi)
                assert torch.equal(o1, o2)


def test_warp_pipelined_kernel_refuses_what_it_cannot_run_and_tune_picks_a_working_kernel(env):
    B = env.B
    for dims, layout in [((32, 4, 4, 4), "aos"), ((16, 4, 4, 4), "soa"), ((64, 4, 2, 2), "soa")]:
        with env.device.Lattice(dims, "f64", layout, False) as lat:
            lat.set_kernel("wpipe")
            o, p, g = lat.new_spinor(), lat.new_spinor(), lat.new_gauge()
            assert B.dslash_apply_status(lat.ctx, o.data_ptr(), p.data_ptr(), g.data_ptr()) == B.DSLASH_ERR_UNSUPPORTED, (dims, layout)
    with env.device.Lattice((32, 4, 4, 4), "f64", "soa", False) as lat:
        for opt, bad in [(B.DSLASH_OPT_PIPE_SLOTS, 1), (B.DSLASH_OPT_PIPE_SLOTS, 5), (B.DSLASH_OPT_PIPE_WARPS, 3), (B.DSLASH_OPT_PIPE_ZBLOCK, 3)]:
            with pytest.raises(B.DslashError):
                B.dslash_set_option(lat.ctx, opt, bad)
    # dslash_tune: times direct (+ wpipe where eligible), keeps one of them, leaves D in in `out`
    for dims, eligible in [((32, 8, 8, 8), True), ((16, 8, 8, 8), False)]:
        g, p, ref, _ = fields_and_ref(env, dims, SEED + 24, "f64")
        with env.device.Lattice(dims, "f64", "soa", False) as lat:
            gi, pi, o = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
            kernel, ms = lat.tune(o, pi, gi)
            assert kernel in ((B.DSLASH_KERNEL_DIRECT, B.DSLASH_KERNEL_WARP_PIPE) if eligible else (B.DSLASH_KERNEL_DIRECT,)) and ms > 0
            assert B.dslash_get_kernel(lat.ctx) == kernel
            assert env.checks.parity_error(lat.download_spinor(o), ref) <= TOL["f64"]
            o.zero_()
            lat.apply(o, pi, gi)
            assert env.checks.parity_error(lat.download_spinor(o), ref) <= TOL["f64"]
            B.dslash_set_option(lat.ctx, B.DSLASH_OPT_TUNE_MODE, B.DSLASH_TUNE_SUSTAINED)
            assert B.dslash_get_option(lat.ctx, B.DSLASH_OPT_TUNE_MODE) == B.DSLASH_TUNE_SUSTAINED
            kernel, ms = lat.tune(o, pi, gi)
            assert kernel in (B.DSLASH_KERNEL_DIRECT, B.DSLASH_KERNEL_WARP_PIPE) and ms > 0
            assert env.checks.parity_error(lat.download_spinor(o), ref) <= TOL["f64"]
            with pytest.raises(B.DslashError):
                B.dslash_set_option(lat.ctx, B.DSLASH_OPT_TUNE_MODE, 2)
            B.dslash_set_variant(lat.ctx, 4, 128, 1)
            assert B.dslash_tune_status(lat.ctx, o.data_ptr(), pi.data_ptr(), gi.data_ptr()) == B.DSLASH_ERR_UNSUPPORTED
    assert B.dslash_tune_status(None, 16, 32, 48) == B.DSLASH_ERR_NULL


# ---------------------------------------------------------------- config 2: 16^4 FP64
@pytest.mark.parametrize("layout,recon12", ALL_MODES)
def test_config2_16x16x16x16(env, layout, recon12):
    dims = (16, 16, 16, 16)
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 2, "f64")
    with env.device.Lattice(dims, "f64", layout, recon12) as lat:
        assert gpu_vs_ref(env, lat, g, p, ref) <= TOL["f64"]


# ---------------------------------------------------------------- config 5: all 120 sweep variants on 24^4 FP64
def test_config5_all_120_variants_24x24x24x24(env):
    dims = (24, 24, 24, 24)
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 5, "f64")
    torch = env.torch
    ref_t = torch.from_numpy(np.ascontiguousarray(ref)).cuda()
    ref_c = torch.view_as_complex(ref_t)
    rms = torch.sqrt(torch.mean(ref_c.abs() ** 2))
    den = torch.maximum(ref_c.abs(), rms)
    lats = {}
    worst = 0.0
    try:
        for lay in ("aos", "soa"):
            lat = env.device.Lattice(dims, "f64", lay, False)
            lats[lay] = (lat, lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor(),
                         lat._bytes(env.B.dslash_canonical_spinor_bytes(lat.ctx)))
        for i in range(env.B.dslash_variant_count()):
            depth, tpb, spt, layout = env.B.dslash_variant_at(i)
            lat, gi, pi, o, can = lats["aos" if layout == env.B.DSLASH_AOS else "soa"]
            o.zero_()
            lat.set_variant(depth, tpb, spt)
            lat.apply(o, pi, gi)
            env.B.dslash_unpack_spinor(lat.ctx, can.data_ptr(), o.data_ptr(), lat.stream())
            got_c = torch.view_as_complex(can.view(torch.float64).view(ref_t.shape))
            e = float(((got_c - ref_c).abs() / den).max())  # same metric as checks.parity_error
            assert e <= TOL["f64"], (depth, tpb, spt, layout, e)
            worst = max(worst, e)
        # and one variant through the NumPy metric, so the torch restatement above is itself checked
        lat, gi, pi, o, can = lats["soa"]
        lat.set_variant(4, 128, 1)
        lat.apply(o, pi, gi)
        e_np = env.checks.parity_error(lat.download_spinor(o), ref)
        assert e_np <= TOL["f64"] and e_np > 0.0
    finally:
        for lat, *_ in lats.values():
            lat.close()


# ---------------------------------------------------------------- the paper's own 84-variant space (42 kernels x 2 map modes)
@pytest.mark.parametrize("dims", [(4, 6, 8, 10), (3, 5, 2, 7)])
def test_all_omp_style_variants_match_the_oracle(env, dims):
    B = env.B
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 15, "f64")
    structures = set()
    for i in range(B.dslash_omp_variant_count(4)):
        x, a, b, sched, _mode = B.dslash_omp_variant_at(4, i)
        structures.add((x, a, b, sched))
    assert len(structures) == 42
    for layout in ("soa", "aos"):
        with env.device.Lattice(dims, "f64", layout, False) as lat:
            gi, pi, o = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
            for (x, a, b, sched) in sorted(structures):
                for teams, team_size in ((0, 128), (3, 32), (7, 256)):
                    B.dslash_set_omp_variant(lat.ctx, x, a, b, sched, teams, team_size)
                    o.zero_()
                    lat.apply(o, pi, gi)
                    e = env.checks.parity_error(lat.download_spinor(o), ref)
                    assert e <= TOL["f64"], (layout, x, a, b, sched, teams, team_size, e)
            for bad in [(0, 1, 1, 0), (1, 0, 1, 0), (1, 2, 1, 0), (2, 1, 3, 0), (4, 1, 1, 0), (0, 0, 5, 0), (0, 0, 1, 3)]:
                with pytest.raises(B.DslashError):
                    B.dslash_set_omp_variant(lat.ctx, *bad)
            with pytest.raises(B.DslashError):
                B.dslash_set_omp_variant(lat.ctx, 0, 0, 4, 0, 0, 48)
            lat.set_variant(B.DSLASH_VARIANT_TUNED)
            assert env.checks.parity_error(lat.dslash(g, p), ref) <= TOL["f64"]


# ---------------------------------------------------------------- operators around Dslash: D^dagger, M, M^dagger, CG
@pytest.mark.parametrize("dims", [(4, 6, 8, 10), (3, 5, 2, 7), (32, 4, 2, 4)])
@pytest.mark.parametrize("precision", ["f64", "f32"])
@pytest.mark.parametrize("layout,recon12", ALL_MODES)
def test_apply_op_matches_the_oracle(env, dims, precision, layout, recon12):
    B = env.B
    g, p = env.inputs.fields(dims, SEED + 16, precision)
    g64, p64 = env.inputs.promote(g), env.inputs.promote(p)
    mass = -0.3
    refs = {B.DSLASH_OP_D: env.oracle.dslash(p64, g64, dims), B.DSLASH_OP_D_DAGGER: env.oracle.dslash_dagger(p64, g64, dims),
            B.DSLASH_OP_M: env.oracle.wilson(p64, g64, dims, mass), B.DSLASH_OP_M_DAGGER: env.oracle.wilson(p64, g64, dims, mass, dagger=True)}
    with env.device.Lattice(dims, precision, layout, recon12) as lat:
        gi, pi, o = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
        for op, ref in refs.items():
            o.zero_()
            lat.apply_op(op, mass, o, pi, gi)
            assert env.checks.parity_error(lat.download_spinor(o), ref) <= TOL[precision], op
        assert B.dslash_apply_status(lat.ctx, o.data_ptr(), pi.data_ptr(), gi.data_ptr()) == B.DSLASH_OK
        with pytest.raises(B.DslashError) as e:
            B.dslash_apply_op(lat.ctx, 4, 0.0, o.data_ptr(), pi.data_ptr(), gi.data_ptr())
        assert e.value.status == B.DSLASH_ERR_UNSUPPORTED
        with pytest.raises(B.DslashError) as e:
            B.dslash_apply_op(lat.ctx, 0, 0.0, pi.data_ptr(), pi.data_ptr(), gi.data_ptr())
        assert e.value.status == B.DSLASH_ERR_ALIAS


@pytest.mark.parametrize("dims,precision,layout,tol", [((8, 8, 8, 8), "f64", "soa", 1e-10), ((6, 4, 10, 5), "f64", "aos", 1e-10),
                                                       ((8, 8, 8, 8), "f32", "soa", 1e-5)])
def test_cg_solves_the_normal_equations(env, dims, precision, layout, tol):
    """x = CG(M^dagger M, b): the residual |M^dagger M x - b| / |b| is evaluated independently with the fp64 oracle."""
    B = env.B
    g, b = env.inputs.fields(dims, SEED + 17, precision)
    g64, b64 = env.inputs.promote(g), env.inputs.promote(b)
    mass = 0.2
    with env.device.Lattice(dims, precision, layout, False) as lat:
        gi, bi, x = lat.upload_gauge(g), lat.upload_spinor(b), lat.new_spinor()
        n0 = B.dslash_launch_count(lat.ctx)
        iters, rel = lat.cg_solve(x, bi, gi, mass, tol, 500)
        assert 1 <= iters < 500 and rel <= tol
        assert B.dslash_launch_count(lat.ctx) >= n0 + 7 * (iters - 1)
        xs = env.inputs.promote(lat.download_spinor(x))
        mx = env.oracle.wilson(xs, g64, dims, mass)
        mdmx = env.oracle.wilson(mx, g64, dims, mass, dagger=True)
        res = np.linalg.norm(mdmx - b64.reshape(mdmx.shape)) / np.linalg.norm(b64)
        assert res <= (5 * tol if precision == "f64" else 5e-5), res
        # b is not modified, a second solve reproduces the first bit for bit (deterministic reductions)
        assert np.array_equal(lat.download_spinor(bi), b)
        x2 = lat.new_spinor()
        iters2, rel2 = lat.cg_solve(x2, bi, gi, mass, tol, 500)
        assert (iters2, rel2) == (iters, rel) and np.array_equal(lat.download_spinor(x2), lat.download_spinor(x))
        # max_iter reached is reported, not an error
        it3, rel3 = lat.cg_solve(x2, bi, gi, mass, 1e-30, 3)
        assert it3 == 3 and rel3 > 1e-30
        for bad in [dict(tol=0.0, max_iter=10), dict(tol=1e-8, max_iter=0)]:
            with pytest.raises(B.DslashError) as e:
                lat.cg_solve(x2, bi, gi, mass, bad["tol"], bad["max_iter"])
            assert e.value.status == B.DSLASH_ERR_UNSUPPORTED


# ---------------------------------------------------------------- multi-GPU slab decomposition, ranks emulated in one process
@pytest.mark.parametrize("world", [1, 2, 3, 4, 6, 12])
@pytest.mark.parametrize("precision,layout,recon12", [("f64", "soa", False), ("f64", "aos", True), ("f32", "soa", True),
                                                      ("f32", "aos", False)])
def test_slab_decomposition_reproduces_the_single_lattice_result(env, world, precision, layout, recon12):
    """T-slabs + half-spinor faces (dslash_slab_pack_faces / _interior / _boundary) must give the oracle's result for the
    GLOBAL lattice, and the same bits as dslash_apply on one GPU.  world = 6 and 12 are the slabs of two and one slices
    (no interior).  One GPU is available, so the ranks are emulated in one process and the exchange is a device copy
    between their face buffers (slab.exchange_faces_in_process); the torch.distributed path is covered on CPU by
    tests/test_multirank_gloo.py."""
    from paper_2301_03636_b200 import slab
    B = env.B
    dims = (8, 4, 4, 12)
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 18, precision)
    with env.device.Lattice(dims, precision, layout, recon12) as lat:
        single = lat.dslash(g, p)
    ranks = [slab.SlabDslash(dims, precision, layout, recon12, rank=r, world=world) for r in range(world)]
    try:
        gauges = [rk.upload_gauge(g) for rk in ranks]
        ins = [rk.upload_spinor(p) for rk in ranks]
        outs = [rk.lat.new_spinor() for rk in ranks]
        for o in outs:
            o.fill_(0x7f)
        # half of a spinor slice per face: 6 complex per site
        rb = 8 if precision == "f64" else 4
        assert ranks[0].face_bytes == dims[0] * dims[1] * dims[2] * 12 * rb and ranks[0].halo_bytes_per_application == 2 * ranks[0].face_bytes
        st = env.torch.cuda.current_stream().cuda_stream
        # the three phases rank by rank, the exchange (for everybody at once) between packing and the boundary slices
        for rk, i, gg in zip(ranks, ins, gauges):
            f = rk.faces
            B.dslash_slab_pack_faces(rk.lat.ctx, f["face_down"].data_ptr(), f["face_up"].data_ptr(), i.data_ptr(), gg.data_ptr(), st)
        slab.exchange_faces_in_process([rk.faces for rk in ranks], [rk.geom for rk in ranks])
        for rk, o, i, gg in zip(ranks, outs, ins, gauges):
            n0 = B.dslash_launch_count(rk.lat.ctx)
            B.dslash_slab_interior(rk.lat.ctx, o.data_ptr(), i.data_ptr(), gg.data_ptr(), st)
            assert B.dslash_launch_count(rk.lat.ctx) == n0 + (1 if rk.geom.lt > 2 else 0)
            f = rk.faces
            B.dslash_slab_boundary(rk.lat.ctx, o.data_ptr(), i.data_ptr(), gg.data_ptr(), f["face_from_below"].data_ptr(),
                                   f["face_from_above"].data_ptr(), st)
        env.torch.cuda.synchronize()
        got = np.concatenate([rk.download(o) for rk, o in zip(ranks, outs)], axis=0)
        assert got.shape == ref.shape
        assert env.checks.parity_error(got, ref) <= TOL[precision]
        assert np.array_equal(got, single)  # the same arithmetic in the same order, merely split between ranks
        if world == 1:  # SlabDslash.apply with the self-wrap exchange
            outs[0].fill_(0x7f)
            ranks[0].apply(outs[0], ins[0], gauges[0])
            env.torch.cuda.synchronize()
            assert np.array_equal(ranks[0].download(outs[0]), single)
    finally:
        for rk in ranks:
            rk.close()


def test_slab_calls_check_their_arguments(env):
    B = env.B
    with env.device.Lattice((8, 4, 4, 6), "f64", "soa", False) as lat:
        o, p, g = lat.new_spinor(), lat.new_spinor(), lat.new_gauge()
        fb = B.dslash_slab_face_bytes(lat.ctx)
        f = [env.torch.zeros(fb, dtype=env.torch.uint8, device="cuda") for _ in range(2)]
        for bad in [lambda: B.dslash_slab_pack_faces(lat.ctx, 0, f[1].data_ptr(), p.data_ptr(), g.data_ptr()),
                    lambda: B.dslash_slab_pack_faces(lat.ctx, f[0].data_ptr(), f[0].data_ptr(), p.data_ptr(), g.data_ptr()),
                    lambda: B.dslash_slab_pack_faces(lat.ctx, f[0].data_ptr() + 8, f[1].data_ptr(), p.data_ptr(), g.data_ptr()),
                    lambda: B.dslash_slab_interior(lat.ctx, p.data_ptr(), p.data_ptr(), g.data_ptr()),
                    lambda: B.dslash_slab_boundary(lat.ctx, o.data_ptr(), p.data_ptr(), g.data_ptr(), f[0].data_ptr(), 0)]:
            with pytest.raises(B.DslashError):
                bad()
        B.dslash_set_time_range(lat.ctx, 1, 4)
        with pytest.raises(B.DslashError) as e:
            B.dslash_slab_interior(lat.ctx, o.data_ptr(), p.data_ptr(), g.data_ptr())
        assert e.value.status == B.DSLASH_ERR_UNSUPPORTED


def test_time_range_only_touches_its_slices(env):
    B = env.B
    dims = (8, 4, 4, 6)
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 19, "f64")
    with env.device.Lattice(dims, "f64", "soa", False) as lat:
        gi, pi, o = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
        o.zero_()
        B.dslash_set_time_range(lat.ctx, 2, 5)
        lat.apply(o, pi, gi)
        out = lat.download_spinor(o)
        assert env.checks.parity_error(out[2:5], ref[2:5]) <= TOL["f64"]
        assert np.all(out[:2] == 0) and np.all(out[5:] == 0)
        lat.apply_op(B.DSLASH_OP_D_DAGGER, 0.0, o, pi, gi)
        assert np.all(lat.download_spinor(o)[:2] == 0)
        lat.set_variant(4, 128, 1)
        assert B.dslash_apply_status(lat.ctx, o.data_ptr(), pi.data_ptr(), gi.data_ptr()) == B.DSLASH_ERR_UNSUPPORTED
        lat.set_variant(B.DSLASH_VARIANT_TUNED)
        for bad in [(-1, 3), (3, 3), (2, 7)]:
            with pytest.raises(B.DslashError):
                B.dslash_set_time_range(lat.ctx, *bad)
        B.dslash_set_time_range(lat.ctx, 0, 6)
        assert env.checks.parity_error(lat.dslash(g, p), ref) <= TOL["f64"]


# ---------------------------------------------------------------- config 3: 32^3 x 64 FP64, 18- and 12-real links
# WHOLE lattice against the oracle, for every kernel dslash_tune() can return, in the launch configurations it tries
# (the oracle applies the 2 M-site lattice in well under a second per core-second on the box).
TUNABLE_KERNELS = [("direct", 0, 0), ("march", 0, 0), ("wpipe", 2, 4), ("wpipe", 3, 1), ("wpipe", 2, 1)]


@pytest.mark.parametrize("recon12", [False, True])
def test_config3_32x32x32x64_fp64(env, recon12):
    B = env.B
    dims = (32, 32, 32, 64)
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 3, "f64", full=True)
    with env.device.Lattice(dims, "f64", "soa", recon12) as lat:
        gi, pi, o = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
        first = None
        for kernel, slots, warps in TUNABLE_KERNELS:
            lat.set_kernel(kernel)
            if kernel == "wpipe":
                B.dslash_set_option(lat.ctx, B.DSLASH_OPT_PIPE_SLOTS, slots)
                B.dslash_set_option(lat.ctx, B.DSLASH_OPT_PIPE_WARPS, warps)
            o.fill_(0x7f)
            lat.apply(o, pi, gi)
            got = lat.download_spinor(o)
            assert env.checks.parity_error(got, ref) <= TOL["f64"], (kernel, slots, warps)
            if first is None:
                first = got
            else:
                assert np.array_equal(got, first), (kernel, slots, warps)  # every tuned kernel gives the same bits
        # and whatever dslash_tune() picks, in both regimes, on the buffer it leaves behind
        for mode in (B.DSLASH_TUNE_BURST, B.DSLASH_TUNE_SUSTAINED):
            B.dslash_set_option(lat.ctx, B.DSLASH_OPT_TUNE_MODE, mode)
            o.fill_(0x7f)
            chosen, ms = B.dslash_tune(lat.ctx, o.data_ptr(), pi.data_ptr(), gi.data_ptr(), lat.stream())
            assert chosen in (B.DSLASH_KERNEL_DIRECT, B.DSLASH_KERNEL_MARCH, B.DSLASH_KERNEL_WARP_PIPE) and ms > 0
            assert np.array_equal(lat.download_spinor(o), first), (mode, chosen)
    _FIELD_CACHE.clear()


def test_config3_full_size_properties(env):
    """Properties that hold at any size, on the bench configuration: unit gauge + constant spinor
    gives 8 psi everywhere; translation of all fields by one site translates the result."""
    dims = (32, 32, 32, 64)
    lx, ly, lz, lt = dims
    chi = np.random.default_rng(3).standard_normal((4, 3, 2))
    psi = np.broadcast_to(chi, (lt, lz, ly, lx, 4, 3, 2))
    u = np.zeros((lt, lz, ly, lx, 4, 3, 3, 2))
    u[..., range(3), range(3), 0] = 1.0
    with env.device.Lattice(dims, "f64", "soa", False) as lat:
        out = lat.dslash(u, psi)
        assert np.abs(out - 8.0 * psi).max() <= 1e-13


def test_config3_staged_kernels_are_bit_stable_under_back_to_back_launches(env):
    """At the bench size, in the bench's launch pattern (back-to-back applications, no host synchronisation in between), every
    tenth result of 200 launches of each staged kernel equals the direct kernel's bit for bit: the hand-offs of the marching
    and warp-pipelined kernels (mbarriers, async-proxy refills, row counters) leave no window in which a slot is overwritten
    early -- the class of fault round 1 found only on a small lattice (one wrong row in 9 % of the launches)."""
    torch = env.torch
    dims = (32, 32, 32, 64)
    with env.device.Lattice(dims, "f64", "soa", False) as lat:
        g, p, ref = lat.new_gauge(), lat.new_spinor(), lat.new_spinor()
        gen = torch.Generator(device=g.device).manual_seed(SEED + 77)
        g.view(torch.float64).normal_(generator=gen)   # bit-stability does not need SU(3) links
        p.view(torch.float64).normal_(generator=gen)
        lat.apply(ref, p, g)
        torch.cuda.synchronize()
        for kernel in ("march", "wpipe"):
            lat.set_kernel(kernel)
            o = lat.new_spinor()
            bad = 0
            for i in range(200):
                lat.apply(o, p, g)
                if i % 10 == 9:
                    torch.cuda.synchronize()
                    bad += 0 if torch.equal(o, ref) else 1
                    o.fill_(0x7f)
            assert bad == 0, kernel


# ---------------------------------------------------------------- the largest lattice the 32-bit site index allows
def test_maximum_lattice_size(env):
    """32 x 128 x 112 x 128 = 58 720 256 sites, FP32: 36 V = 2 113 929 216 < 2^31 is the limit dslash_create enforces
    (dims one step larger are refused).  No oracle run fits this size, so the check is a property that holds at any size and is
    sensitive to every neighbour index: with unit links and psi(x) = s(x) chi (s a random real field, chi one spinor), Eq. 1
     gives  D psi(x) = [sum_mu s(x+mu) + s(x-mu)] chi - sum_mu [s(x+mu) - s(x-mu)] gamma_mu chi,  evaluated here
    with torch.roll and the oracle's gamma matrices.  Then, on random links and spinors, the marching and warp-pipelined
    kernels (plan- and row-based addressing) must give the direct kernel's bits."""
    torch, B = env.torch, env.B
    dims = (32, 128, 112, 128)
    lx, ly, lz, lt = dims
    v = lx * ly * lz * lt
    with pytest.raises(B.DslashError):
        B.dslash_create((32, 128, 114, 128), B.DSLASH_FP32, B.DSLASH_SOA)
    dev = torch.device("cuda:0")
    gen = torch.Generator(device=dev).manual_seed(SEED + 58)
    rng = np.random.default_rng(SEED + 58)
    chi = rng.standard_normal(12) + 1j * rng.standard_normal(12)          # index = spin * 3 + colour
    gchi = [np.einsum("ab,bc->ac", env.oracle.gamma(mu), chi.reshape(4, 3)).reshape(12) for mu in range(4)]
    to_ri = lambda z: torch.from_numpy(np.stack([z.real, z.imag], -1)).to(dev)   # [12, 2] float64
    chi_t, gchi_t = to_ri(chi), [to_ri(z) for z in gchi]
    s = torch.randn((lt, lz, ly, lx), generator=gen, device=dev, dtype=torch.float64)
    with env.device.Lattice(dims, "f32", "soa", False) as lat:
        st = lat.stream()
        # inputs in the canonical layout on the device, packed by the library
        can = (s[..., None, None] * chi_t).to(torch.float32).contiguous()                      # [T,Z,Y,X,12,2]
        p = lat.new_spinor()
        B.dslash_pack_spinor(lat.ctx, p.data_ptr(), can.data_ptr(), st)
        del can
        u = torch.zeros((v, 4, 3, 3, 2), device=dev, dtype=torch.float32)
        u[:, :, range(3), range(3), 0] = 1.0
        g = lat.new_gauge()
        B.dslash_pack_gauge(lat.ctx, g.data_ptr(), u.data_ptr(), st)
        torch.cuda.synchronize()
        del u
        o = lat.new_spinor()
        o.fill_(0x7f)
        lat.apply(o, p, g)
        out = torch.empty((lt, lz, ly, lx, 12, 2), device=dev, dtype=torch.float32)
        B.dslash_unpack_spinor(lat.ctx, out.data_ptr(), o.data_ptr(), st)
        torch.cuda.synchronize()
        # expected, slab by slab in t (fp64)
        shift = {0: 3, 1: 2, 2: 1, 3: 0}   # axis of direction mu in [T,Z,Y,X]
        fwd = [torch.roll(s, -1, shift[mu]) for mu in range(4)]
        bwd = [torch.roll(s, +1, shift[mu]) for mu in range(4)]
        a = sum(fwd) + sum(bwd)
        err2 = 0.0
        ref2 = 0.0
        worst = 0.0
        for t0 in range(0, lt, 8):
            sl = slice(t0, t0 + 8)
            exp = a[sl][..., None, None] * chi_t
            for mu in range(4):
                exp = exp - (fwd[mu][sl] - bwd[mu][sl])[..., None, None] * gchi_t[mu]
            d = out[sl].to(torch.float64) - exp
            worst = max(worst, float(d.abs().max()))
            ref2 += float((exp * exp).sum())
        rms = (ref2 / (v * 12)) ** 0.5          # rms magnitude of a complex component
        assert worst / rms <= TOL["f32"], (worst, rms)
        del out, fwd, bwd, a, s
        # random links and spinors: three independent addressing schemes, the same bits
        g.view(torch.float32).normal_(generator=gen)
        p.view(torch.float32).normal_(generator=gen)
        lat.apply(o, p, g)
        torch.cuda.synchronize()
        for kernel in ("march", "wpipe"):
            lat.set_kernel(kernel)
            o2 = lat.new_spinor()
            o2.fill_(0x7f)
            lat.apply(o2, p, g)
            torch.cuda.synchronize()
            assert torch.equal(o2, o), kernel
            del o2


# ---------------------------------------------------------------- config 4: 48^3 x 96 FP32 vs the FP64 oracle
def test_config4_48x48x48x96_fp32(env):
    """WHOLE lattice (10.6 M sites) against the fp64 oracle; dslash_tune() first, so the kernel checked is the one bench.py times."""
    B = env.B
    dims = (48, 48, 48, 96)
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 4, "f32", full=True)
    with env.device.Lattice(dims, "f32", "soa", False) as lat:
        gi, pi, o = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
        o.fill_(0x7f)
        lat.apply(o, pi, gi)
        direct = lat.download_spinor(o)
        assert env.checks.parity_error(direct, ref) <= TOL["f32"]
        del ref
        _FIELD_CACHE.clear()
        o.fill_(0x7f)
        chosen, _ = B.dslash_tune(lat.ctx, o.data_ptr(), pi.data_ptr(), gi.data_ptr(), lat.stream())
        assert np.array_equal(lat.download_spinor(o), direct), chosen


# ---------------------------------------------------------------- invariants evaluated on the GPU itself
def test_gpu_gauge_covariance_and_translation(env):
    dims = (6, 4, 8, 10)
    v = int(np.prod(dims))
    g, p = env.inputs.fields(dims, SEED + 21)
    gc = g[..., 0] + 1j * g[..., 1]
    pc = p[..., 0] + 1j * p[..., 1]
    G = env.inputs.haar_su3(v, np.random.default_rng(5)).reshape(dims[3], dims[2], dims[1], dims[0], 3, 3)
    ug = np.empty_like(gc)
    for mu in range(4):
        ug[..., mu, :, :] = G @ gc[..., mu, :, :] @ np.conj(np.swapaxes(np.roll(G, -1, axis=3 - mu), -1, -2))
    pg = np.einsum("tzyxij,tzyxaj->tzyxai", G, pc)
    c2r = lambda a: np.ascontiguousarray(np.stack([a.real, a.imag], axis=-1))
    with env.device.Lattice(dims, "f64", "soa", False) as lat:
        lhs = lat.dslash(c2r(ug), c2r(pg))
        rhs = lat.dslash(g, p)
        rhs_c = np.einsum("tzyxij,tzyxaj->tzyxai", G, rhs[..., 0] + 1j * rhs[..., 1])
        assert env.checks.parity_error(lhs, c2r(rhs_c)) <= 1e-12
        for mu in range(4):
            ax = 3 - mu
            rolled = lat.dslash(np.roll(g, 1, axis=ax), np.roll(p, 1, axis=ax))
            assert np.array_equal(rolled, np.roll(rhs, 1, axis=ax))  # same arithmetic, bit for bit


# ---------------------------------------------------------------- layout module round trip
@pytest.mark.parametrize("precision", ["f64", "f32"])
@pytest.mark.parametrize("layout", ["aos", "soa"])
@pytest.mark.parametrize("dims", [(8, 4, 3, 4), (5, 4, 3, 6)])  # V a multiple of 32 / a ragged last vector
def test_pack_unpack_round_trip_is_bit_exact(env, precision, layout, dims):
    g, p = env.inputs.fields(dims, SEED + 31, precision)
    with env.device.Lattice(dims, precision, layout, False) as lat:
        back = lat.download_spinor(lat.upload_spinor(p))
        assert np.array_equal(back, p)
        nat = lat.upload_gauge(g).cpu().numpy().view(lat.np_dtype)
        v = lat.volume
        assert np.array_equal(nat[:soa_ref(g.reshape(v, 36, 2), layout).size], soa_ref(g.reshape(v, 36, 2), layout))
    with env.device.Lattice(dims, precision, layout, True) as lat:
        nat = lat.upload_gauge(g).cpu().numpy().view(lat.np_dtype)
        g12 = np.ascontiguousarray(g.reshape(v, 4, 3, 3, 2)[:, :, :2]).reshape(v, 24, 2)
        assert np.array_equal(nat[:soa_ref(g12, layout).size], soa_ref(g12, layout))
        ps = lat.upload_spinor(p).cpu().numpy().view(lat.np_dtype)
        pref = soa_ref(p.reshape(v, 12, 2), layout)
        assert np.array_equal(ps[:pref.size], pref)


def soa_ref(a, layout):
    """Reference native image of a canonical [V, ncomp, 2] field (NumPy, layout arithmetic only).
    soa: blocked SoA of include/dslash_b200.h -- [ceil(V/32)][ncomp][32][2] for 16-byte (fp64) or 8-byte (fp32
    link) elements; fp32 spinors pair components (2q, 2q+1) into float4 units: [v][6][32][4].  The last
    vector is compared only up to the last real site."""
    v, nc, _ = a.shape
    if layout == "aos":
        return a.reshape(-1)
    nv = (v + 31) // 32
    pad = np.zeros((nv * 32, nc, 2), dtype=a.dtype)
    pad[:v] = a
    if a.dtype == np.float32 and nc == 12:  # fp32 spinor: float4 units
        out = pad.reshape(nv, 32, 6, 4).transpose(0, 2, 1, 3)
    else:
        out = pad.reshape(nv, 32, nc, 2).transpose(0, 2, 1, 3)
    flat = np.ascontiguousarray(out).reshape(-1)
    # drop the (unspecified) padding tail: keep whole vectors only if V is a multiple of 32
    if v % 32:
        full = (v // 32) * 32 * nc * 2
        return flat[:full]
    return flat


# ---------------------------------------------------------------- error behaviour on a live context
def test_error_paths_on_device(env):
    B = env.B
    with env.device.Lattice((4, 4, 4, 4), "f64", "soa", False) as lat:
        o, p, g = lat.new_spinor(), lat.new_spinor(), lat.new_gauge()
        assert B.dslash_apply_status(lat.ctx, o.data_ptr() + 8, p.data_ptr(), g.data_ptr()) == B.DSLASH_ERR_ALIGN
        assert B.dslash_apply_status(lat.ctx, p.data_ptr(), p.data_ptr(), g.data_ptr()) == B.DSLASH_ERR_ALIAS
        assert B.dslash_apply_status(lat.ctx, p.data_ptr() + 16, p.data_ptr(), g.data_ptr()) == B.DSLASH_ERR_ALIAS
        assert B.dslash_apply_status(lat.ctx, 0, p.data_ptr(), g.data_ptr()) == B.DSLASH_ERR_NULL
        for bad in [(5, 64, 1), (4, 96, 1), (4, 64, 3), (-1, 64, 1)]:
            with pytest.raises(B.DslashError) as e:
                lat.set_variant(*bad)
            assert e.value.status == B.DSLASH_ERR_UNSUPPORTED
        for bad in [(3, 4, 4, 4), (64, 32, 1, 1), (1, 1, 1, 1), (0, 4, 4, 4)]:
            with pytest.raises(B.DslashError) as e:
                lat.set_tile(bad)
            assert e.value.status == B.DSLASH_ERR_UNSUPPORTED
        lat.set_variant(3, 256, 2)
        assert B.dslash_get_variant(lat.ctx) == (3, 256, 2)
        lat.set_variant(B.DSLASH_VARIANT_TUNED)
        assert B.dslash_get_variant(lat.ctx)[0] == B.DSLASH_VARIANT_TUNED
        assert B.dslash_last_cuda_error(lat.ctx) == 0


# ---------------------------------------------------------------- host entry point (e2e path) and its byte accounting
@pytest.mark.parametrize("layout,recon12", [("soa", False), ("soa", True), ("aos", False)])
@pytest.mark.parametrize("dims,precision", [
    ((8, 6, 4, 10), "f64"),   # 10 slabs of one time slice (192 sites = 6 vectors) pipelined over three streams
    ((32, 4, 4, 40), "f64"),  # 32 slabs of 1-2 slices
    ((32, 4, 4, 40), "f32"),
    ((6, 3, 5, 4), "f64"),    # a slice of 90 sites is not a whole number of vectors: blocked SoA runs as one slab, AoS as 4
    ((4, 4, 4, 2), "f64"),    # two slabs: each one's neighbours in t are both the other one
    ((4, 4, 2, 1), "f64"),    # a single time slice
])
def test_apply_host_matches_oracle_and_counts_bytes(env, layout, recon12, dims, precision):
    g, p, ref, _ = fields_and_ref(env, dims, SEED + 41, precision)
    torch, B = env.torch, env.B
    gh = torch.from_numpy(g.copy()).pin_memory()
    ph = torch.from_numpy(p.copy()).pin_memory()
    oh = torch.zeros(p.shape, dtype=ph.dtype).pin_memory()
    with env.device.Lattice(dims, precision, layout, recon12) as lat:
        h2d, d2h = B.dslash_apply_host(lat.ctx, oh.data_ptr(), ph.data_ptr(), gh.data_ptr(), B.DSLASH_MAP_MINIMAL, lat.stream())
        assert env.checks.parity_error(oh.numpy(), ref) <= TOL[precision]
        assert (h2d, d2h) == (g.nbytes + p.nbytes, p.nbytes)  # every byte crosses the host link once
        # the same field, bit for bit, as the device-resident path
        assert np.array_equal(oh.numpy(), lat.dslash(g, p))
        # on a side stream, twice in a row (the internal streams are ordered after the caller's stream)
        st = torch.cuda.Stream()
        oh.zero_()
        B.dslash_apply_host(lat.ctx, oh.data_ptr(), ph.data_ptr(), gh.data_ptr(), B.DSLASH_MAP_MINIMAL, st.cuda_stream)
        B.dslash_apply_host(lat.ctx, oh.data_ptr(), ph.data_ptr(), gh.data_ptr(), B.DSLASH_MAP_MINIMAL, st.cuda_stream)
        assert env.checks.parity_error(oh.numpy(), ref) <= TOL[precision]
        oh.zero_()
        h2d2, d2h2 = B.dslash_apply_host(lat.ctx, oh.data_ptr(), ph.data_ptr(), gh.data_ptr(), B.DSLASH_MAP_TOFROM, lat.stream())
        assert env.checks.parity_error(oh.numpy(), ref) <= TOL[precision]
        # PAPER.md:265 (Fig. 4): 1.5 GB without data analysis -> 0.75 GB with it, exactly 2:1
        assert h2d2 + d2h2 == 2 * (h2d + d2h)
        assert np.array_equal(gh.numpy(), g) and np.array_equal(ph.numpy(), p)


# ---------------------------------------------------------------- the probe kernels (bench.py --probe) do what they say
def test_probe_kernels_move_the_bytes_they_claim(env):
    B, torch = env.B, env.torch
    dev = torch.device("cuda:0")
    n = 100003  # 16-byte units, not a multiple of anything
    src = torch.randn(4 * n * 2, dtype=torch.float64, device=dev)
    dst = torch.zeros(n * 2, dtype=torch.float64, device=dev)
    st = torch.cuda.current_stream().cuda_stream
    B.dslash_probe_launch(B.DSLASH_PROBE_COPY, dst.data_ptr(), src.data_ptr(), n, 37, st)
    assert torch.equal(dst, src[:2 * n])
    B.dslash_probe_launch(B.DSLASH_PROBE_READ4_WRITE1, dst.data_ptr(), src.data_ptr(), n, 37, st)
    want = ((src[:2 * n] + src[2 * n:4 * n]) + src[4 * n:6 * n]) + src[6 * n:]
    assert torch.equal(dst, want)
    B.dslash_probe_launch(B.DSLASH_PROBE_WRITE, dst.data_ptr(), 0, n, 37, st)
    assert torch.equal(dst.view(n, 2), torch.tensor([1.0, 2.0], dtype=torch.float64, device=dev).expand(n, 2))
    keep = dst.clone()
    B.dslash_probe_launch(B.DSLASH_PROBE_READ, dst.data_ptr(), src.data_ptr(), 4 * n, 37, st)
    B.dslash_probe_launch(B.DSLASH_PROBE_DFMA, dst.data_ptr(), 0, 100, 37, st)
    torch.cuda.synchronize()
    assert torch.equal(dst, keep)  # the read and FMA probes never write

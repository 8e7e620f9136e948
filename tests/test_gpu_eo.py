"""GPU parity of the even-odd (checkerboarded) path against the oracle's definitions (oracle.dslash_parity,
oracle.schur_even, oracle.wilson), through the C ABI.  Tolerances as in test_gpu_parity.py.

The CUDA side never sees a full-lattice operator here: fields travel as checkerboard halves, so a wrong half-index,
parity offset or gauge half shows up as an O(1) error against the oracle, which works on full-lattice arrays with masks.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-5}
SEED = 230103636
ALL_MODES = [(lay, r12) for lay in ("aos", "soa") for r12 in (False, True)]


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


def masked(env, a, dims, parity):
    odd = env.oracle.parity_mask(dims)
    keep = odd if parity == 1 else ~odd
    return a * keep[..., None, None, None]


# lattices: several tiles + ragged tile edges (12 = 8+4 half-sites in x), L_X = 2 (one half-site per row: x+1 == x-1),
# all-different extents, a half volume that is not a multiple of 32 (padded last SoA vector)
EO_DIMS = [(4, 4, 4, 4), (24, 6, 4, 2), (2, 4, 6, 8), (8, 6, 4, 10), (6, 2, 2, 2), (64, 2, 2, 4), (2, 2, 2, 2)]


@pytest.mark.parametrize("dims", EO_DIMS)
@pytest.mark.parametrize("precision", ["f64", "f32"])
@pytest.mark.parametrize("layout,recon12", ALL_MODES)
def test_eo_dslash_matches_the_oracle_restriction(env, dims, precision, layout, recon12):
    g, p = env.inputs.fields(dims, SEED + 31, precision)
    g64, p64 = env.inputs.promote(g), env.inputs.promote(p)
    with env.device.Lattice(dims, precision, layout, recon12) as lat:
        ge = lat.upload_eo_gauge(g)
        for out_parity in (0, 1):
            pin = lat.upload_eo_spinor(p, 1 - out_parity)
            for dagger in (0, 1):
                ref = env.oracle.dslash_parity(p64, g64, dims, out_parity, bool(dagger))
                out = lat.new_eo_spinor()
                lat.eo_apply(out_parity, dagger, out, pin, ge)
                got = lat.download_eo_spinor({out_parity: out})
                assert env.checks.parity_error(got, ref) <= TOL[precision], (out_parity, dagger)
                # nothing is written on the other parity by the unpack
                assert not masked(env, got, dims, 1 - out_parity).any()


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 6, 4, 10), (24, 6, 4, 2)])
@pytest.mark.parametrize("precision", ["f64", "f32"])
@pytest.mark.parametrize("layout,recon12", ALL_MODES)
def test_eo_schur_complement_matches_the_oracle(env, dims, precision, layout, recon12):
    g, p = env.inputs.fields(dims, SEED + 32, precision)
    g64, p64 = env.inputs.promote(g), env.inputs.promote(p)
    mass = -0.2
    with env.device.Lattice(dims, precision, layout, recon12) as lat:
        ge, pe = lat.upload_eo_gauge(g), lat.upload_eo_spinor(p, 0)
        for dagger in (0, 1):
            ref = env.oracle.schur_even(p64, g64, dims, mass, bool(dagger))
            out, tmp = lat.new_eo_spinor(), lat.new_eo_spinor()
            lat.eo_apply_schur(dagger, mass, out, pe, tmp, ge)
            assert env.checks.parity_error(lat.download_eo_spinor({0: out}), ref) <= TOL[precision], dagger


@pytest.mark.parametrize("precision", ["f64", "f32"])
@pytest.mark.parametrize("layout", ["aos", "soa"])
@pytest.mark.parametrize("dims", [(8, 4, 4, 4), (6, 2, 4, 2)])  # half volume a multiple of 32 / a ragged last vector
def test_eo_pack_unpack_round_trip_is_bit_exact(env, precision, layout, dims):
    g, p = env.inputs.fields(dims, SEED + 33, precision)
    with env.device.Lattice(dims, precision, layout, False) as lat:
        halves = {par: lat.upload_eo_spinor(p, par) for par in (0, 1)}
        assert np.array_equal(lat.download_eo_spinor(halves), p)
        for par in (0, 1):
            assert np.array_equal(lat.download_eo_spinor({par: halves[par]}), masked(env, p, dims, par))
        # the checkerboarded links reproduce the full operator: D psi = D_eo psi_o + D_oe psi_e, against the plain D
        ge = lat.upload_eo_gauge(g)
        outs = {}
        for par in (0, 1):
            outs[par] = lat.new_eo_spinor()
            lat.eo_apply(par, 0, outs[par], halves[1 - par], ge)
        ref = env.oracle.dslash(env.inputs.promote(p), env.inputs.promote(g), dims)
        assert env.checks.parity_error(lat.download_eo_spinor(outs), ref) <= TOL[precision]


@pytest.mark.parametrize("dims,precision,layout,tol", [((8, 8, 8, 8), "f64", "soa", 1e-10), ((6, 4, 10, 4), "f64", "aos", 1e-10),
                                                       ((8, 8, 8, 8), "f32", "soa", 1e-5)])
def test_eo_solve_solves_the_full_wilson_system(env, dims, precision, layout, tol):
    """x from dslash_eo_solve must solve the UNPRECONDITIONED system: |M x - b| / |b| evaluated with the fp64 oracle's
    full-lattice Wilson matrix; and the preconditioned CG needs fewer iterations than the plain one."""
    B = env.B
    g, b = env.inputs.fields(dims, SEED + 34, precision)
    g64, b64 = env.inputs.promote(g), env.inputs.promote(b)
    mass = 0.2
    with env.device.Lattice(dims, precision, layout, False) as lat:
        ge = lat.upload_eo_gauge(g)
        be, bo = lat.upload_eo_spinor(b, 0), lat.upload_eo_spinor(b, 1)
        xe, xo = lat.new_eo_spinor(), lat.new_eo_spinor()
        n0 = B.dslash_launch_count(lat.ctx)
        iters, rel = lat.eo_solve(xe, xo, be, bo, ge, mass, tol, 500)
        assert 1 <= iters < 500 and rel <= tol
        assert B.dslash_launch_count(lat.ctx) >= n0 + 9 * (iters - 1)
        x = env.inputs.promote(lat.download_eo_spinor({0: xe, 1: xo}))
        res = np.linalg.norm(env.oracle.wilson(x, g64, dims, mass) - b64.reshape(x.shape)) / np.linalg.norm(b64)
        assert res <= (20 * tol if precision == "f64" else 1e-4), res
        # b untouched; deterministic
        assert np.array_equal(lat.download_eo_spinor({0: be, 1: bo}), b)
        xe2, xo2 = lat.new_eo_spinor(), lat.new_eo_spinor()
        assert lat.eo_solve(xe2, xo2, be, bo, ge, mass, tol, 500) == (iters, rel)
        assert np.array_equal(lat.download_eo_spinor({0: xe2, 1: xo2}), lat.download_eo_spinor({0: xe, 1: xo}))
        # the plain normal-equation CG on the same M needs more iterations to the same tolerance
        gi, bi, xf = lat.upload_gauge(g), lat.upload_spinor(b), lat.new_spinor()
        iters_plain, _ = lat.cg_solve(xf, bi, gi, mass, tol, 500)
        assert iters < iters_plain, (iters, iters_plain)


def test_eo_cg_solves_the_preconditioned_normal_equations(env):
    dims, mass, tol = (8, 4, 6, 4), 0.1, 1e-10
    g, b = env.inputs.fields(dims, SEED + 35, "f64")
    with env.device.Lattice(dims, "f64", "soa", True) as lat:
        ge, be, xe = lat.upload_eo_gauge(g), lat.upload_eo_spinor(b, 0), lat.new_eo_spinor()
        iters, rel = lat.eo_cg_solve(xe, be, ge, mass, tol, 300)
        assert 1 <= iters < 300 and rel <= tol
        x = lat.download_eo_spinor({0: xe})
        mx = env.oracle.schur_even(x, g, dims, mass)
        mdmx = env.oracle.schur_even(mx, g, dims, mass, dagger=True)
        be_ref = masked(env, b, dims, 0)
        assert np.linalg.norm(mdmx - be_ref) / np.linalg.norm(be_ref) <= 5 * tol
        it3, rel3 = lat.eo_cg_solve(xe, be, ge, mass, 1e-30, 3)
        assert it3 == 3 and rel3 > 1e-30


def test_eo_error_paths(env):
    B = env.B
    with env.device.Lattice((4, 3, 4, 4), "f64", "soa", False) as lat:  # an odd extent: no checkerboard
        assert B.dslash_eo_spinor_bytes(lat.ctx) == 0 and B.dslash_eo_gauge_bytes(lat.ctx) == 0
        buf = lat.new_spinor()
        assert B.dslash_eo_apply_status(lat.ctx, 0, 0, buf.data_ptr(), buf.data_ptr() + 4096, buf.data_ptr()) == B.DSLASH_ERR_DIMS
        with pytest.raises(B.DslashError) as e:
            B.dslash_eo_pack_gauge(lat.ctx, buf.data_ptr(), buf.data_ptr())
        assert e.value.status == B.DSLASH_ERR_DIMS
    with env.device.Lattice((4, 4, 4, 4), "f64", "soa", False) as lat:
        v = 256
        assert B.dslash_eo_spinor_bytes(lat.ctx) == (v // 2) * 24 * 8
        assert B.dslash_eo_gauge_bytes(lat.ctx) == v * 72 * 8
        a, b, g = lat.new_eo_spinor(), lat.new_eo_spinor(), lat._bytes(B.dslash_eo_gauge_bytes(lat.ctx))
        st = B.dslash_eo_apply_status
        assert st(lat.ctx, 0, 0, 0, b.data_ptr(), g.data_ptr()) == B.DSLASH_ERR_NULL
        assert st(lat.ctx, 2, 0, a.data_ptr(), b.data_ptr(), g.data_ptr()) == B.DSLASH_ERR_UNSUPPORTED
        assert st(lat.ctx, 0, 2, a.data_ptr(), b.data_ptr(), g.data_ptr()) == B.DSLASH_ERR_UNSUPPORTED
        assert st(lat.ctx, 0, 0, a.data_ptr() + 8, b.data_ptr(), g.data_ptr()) == B.DSLASH_ERR_ALIGN
        assert st(lat.ctx, 0, 0, a.data_ptr(), a.data_ptr(), g.data_ptr()) == B.DSLASH_ERR_ALIAS
        with pytest.raises(B.DslashError) as e:
            B.dslash_eo_apply_xpay(lat.ctx, 0, 0, a.data_ptr(), b.data_ptr(), g.data_ptr(), a.data_ptr(), 1.0, 1.0)
        assert e.value.status == B.DSLASH_ERR_ALIAS
        with pytest.raises(B.DslashError) as e:
            B.dslash_eo_apply_schur(lat.ctx, 0, -4.0, a.data_ptr(), b.data_ptr(), g.data_ptr(), g.data_ptr())
        assert e.value.status == B.DSLASH_ERR_UNSUPPORTED
        with pytest.raises(B.DslashError) as e:
            B.dslash_eo_cg_solve(lat.ctx, a.data_ptr(), b.data_ptr(), g.data_ptr(), 0.1, 0.0, 10)
        assert e.value.status == B.DSLASH_ERR_UNSUPPORTED
        with pytest.raises(B.DslashError) as e:
            B.dslash_eo_solve(lat.ctx, a.data_ptr(), a.data_ptr(), b.data_ptr(), b.data_ptr(), g.data_ptr(), 0.1, 1e-8, 10)
        assert e.value.status == B.DSLASH_ERR_ALIAS


def test_eo_at_bench_size_sampled(env):
    """32^3x64 fp64 (BASELINE.json configs[2]) in the checkerboarded form, on sampled sites the oracle computes one by one:
    for a source supported on one parity, (D psi)(s) of the plain definition at a site of the other parity IS D_{p,1-p}."""
    dims = (32, 32, 32, 64)
    g, p = env.inputs.fields(dims, SEED + 3, "f64")
    sites = env.inputs.sample_sites(dims, 4096, SEED + 36)
    odd = env.oracle.parity_mask(dims).reshape(-1)
    with env.device.Lattice(dims, "f64", "soa", False) as lat:
        ge = lat.upload_eo_gauge(g)
        for out_parity in (0, 1):
            src = masked(env, p, dims, 1 - out_parity)
            sel = sites[odd[sites] == bool(out_parity)]
            ref = env.oracle.dslash_sites(src, g, dims, sel)
            out = lat.new_eo_spinor()
            lat.eo_apply(out_parity, 0, out, lat.upload_eo_spinor(p, 1 - out_parity), ge)
            got = lat.download_eo_spinor({out_parity: out}).reshape(-1, 4, 3, 2)[sel]
            assert env.checks.parity_error(got, ref) <= TOL["f64"]

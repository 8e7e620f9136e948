"""dslash_eo_apply_schur_static: the Schur operator for callers that cannot allocate device memory.

Who that is: a program that gave the whole GPU to its own memory pool when it started (so a cudaMalloc made inside this library
would fail or eat into that pool), a solver loop that cannot afford the device-wide stall an allocation may cause, or a plug-in
that is handed pointers and owns no device memory at all.  For them the library keeps the operator's odd-parity intermediate in
an 8 MiB array of its own image (include/dslash_b200.h, csrc/dslash_eo.cu) instead of asking for a scratch field.

The check: the new entry point against the existing dslash_eo_apply_schur (caller's scratch field), on two calls in a row that
differ in lattice, precision, layout and input, so the second call finds the first one's data in the shared array.  Both paths
launch the same two kernels on the same data, so the results must be equal bit for bit, which is inside the 1e-12 / 1e-5
relative tolerance the parity tests use (asserted as well).  This file is named to be collected last: it must pass on its own
in a fresh process (its first call is then the per-device set-up) and after every other GPU test.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-5}
SEED = 230103636 + 77
MASS = -0.2


@pytest.fixture(scope="module")
def env():
    import torch
    from paper_2301_03636_b200 import binding, checks, device, inputs
    assert torch.cuda.is_available()

    class E:
        pass
    e = E()
    e.torch, e.B, e.checks, e.device, e.inputs = torch, binding, checks, device, inputs
    return e


def schur_both_ways(env, dims, precision, layout, recon12, dagger, seed, static_first):
    """Returns (static result, existing-path result) as canonical NumPy arrays, and the raw device buffers' equality."""
    g, p = env.inputs.fields(dims, seed, precision)
    with env.device.Lattice(dims, precision, layout, recon12) as lat:
        assert env.B.dslash_eo_spinor_bytes(lat.ctx) <= env.B.dslash_static_scratch_bytes()
        ge, pe = lat.upload_eo_gauge(g), lat.upload_eo_spinor(p, 0)
        out_static, out_ref, tmp = lat.new_eo_spinor(), lat.new_eo_spinor(), lat.new_eo_spinor()
        out_static.fill_(0x7f)  # a site the kernels skip would keep this pattern
        out_ref.fill_(0x7f)
        if static_first:
            lat.eo_apply_schur_static(dagger, MASS, out_static, pe, ge)
            lat.eo_apply_schur(dagger, MASS, out_ref, pe, tmp, ge)
        else:
            lat.eo_apply_schur(dagger, MASS, out_ref, pe, tmp, ge)
            lat.eo_apply_schur_static(dagger, MASS, out_static, pe, ge)
        env.torch.cuda.synchronize()
        same_bytes = bool(env.torch.equal(out_static, out_ref))
        return lat.download_eo_spinor({0: out_static}), lat.download_eo_spinor({0: out_ref}), same_bytes


def test_static_scratch_schur_equals_the_callers_scratch_path_on_two_calls_in_a_row(env):
    # call 1: 16^4 FP64 blocked-SoA (6.3 MB of the 8 MiB array; the largest BASELINE lattice that fits), the static path first
    # call 2: a small ragged lattice (half volume 240 = 7.5 SoA vectors) in FP32 with 12-real links and the adjoint operator:
    #         it reads an array still full of call 1's FP64 data
    calls = [((16, 16, 16, 16), "f64", "soa", False, 0, True),
             ((8, 6, 4, 10), "f32", "soa", True, 1, False)]
    for k, (dims, precision, layout, recon12, dagger, static_first) in enumerate(calls):
        got, ref, same_bytes = schur_both_ways(env, dims, precision, layout, recon12, dagger, SEED + k, static_first)
        assert np.isfinite(ref).all() and np.abs(ref).max() > 0
        assert env.checks.parity_error(got, ref) <= TOL[precision], (k, dims)
        assert same_bytes and np.array_equal(got, ref), (k, dims)


@pytest.mark.parametrize("layout,recon12", [("aos", False), ("soa", True)])
def test_repeated_static_calls_reuse_the_array_and_allocate_nothing(env, layout, recon12):
    dims, precision = (8, 8, 8, 8), "f64"
    g, p = env.inputs.fields(dims, SEED + 5, precision)
    g2, p2 = env.inputs.fields(dims, SEED + 6, precision)
    with env.device.Lattice(dims, precision, layout, recon12) as lat:
        ge, pe, pe2 = lat.upload_eo_gauge(g), lat.upload_eo_spinor(p, 0), lat.upload_eo_spinor(p2, 0)
        tmp = lat.new_eo_spinor()
        ref = [lat.new_eo_spinor(), lat.new_eo_spinor()]
        out = [lat.new_eo_spinor(), lat.new_eo_spinor()]
        lat.eo_apply_schur(0, MASS, ref[0], pe, tmp, ge)
        lat.eo_apply_schur(1, MASS, ref[1], pe2, tmp, ge)
        lat.eo_apply_schur_static(0, MASS, out[0], pe, ge)  # set-up has happened by now at the latest
        env.torch.cuda.synchronize()
        free_before = env.torch.cuda.mem_get_info()[0]
        launches_before = env.B.dslash_launch_count(lat.ctx)
        for _ in range(3):  # back to back on one stream: stream order keeps the calls from sharing the array at the same time
            lat.eo_apply_schur_static(0, MASS, out[0], pe, ge)
            lat.eo_apply_schur_static(1, MASS, out[1], pe2, ge)
        env.torch.cuda.synchronize()
        assert env.torch.cuda.mem_get_info()[0] == free_before  # no device memory was taken
        assert env.B.dslash_launch_count(lat.ctx) == launches_before + 12
        assert env.torch.equal(out[0], ref[0]) and env.torch.equal(out[1], ref[1])


def test_a_field_beyond_the_built_in_array_is_refused_with_its_own_status(env):
    B = env.B
    assert B.dslash_static_scratch_bytes() == B.DSLASH_STATIC_SCRATCH_BYTES == 8 << 20
    ctx = B.dslash_create((24, 24, 24, 24), B.DSLASH_FP64, B.DSLASH_SOA)  # half-lattice spinor 31.9 MB
    try:
        assert B.dslash_eo_spinor_bytes(ctx) > B.dslash_static_scratch_bytes()
        launches = B.dslash_launch_count(ctx)
        assert B.dslash_eo_apply_schur_static_status(ctx, 0, MASS, 16, 32, 48) == B.DSLASH_ERR_TOO_LARGE  # before any launch
        assert B.dslash_launch_count(ctx) == launches
        with pytest.raises(B.DslashError) as e:
            B.dslash_eo_apply_schur_static(ctx, 0, MASS, 16, 32, 48)
        assert e.value.status == B.DSLASH_ERR_TOO_LARGE and "DSLASH_STATIC_SCRATCH_BYTES" in str(e.value)
    finally:
        B.dslash_destroy(ctx)
    ctx = B.dslash_create((16, 16, 16, 16), B.DSLASH_FP64, B.DSLASH_SOA)
    try:  # the other argument checks of the existing entry point apply unchanged
        assert B.dslash_eo_apply_schur_static_status(None, 0, MASS, 16, 32, 48) == B.DSLASH_ERR_NULL
        assert B.dslash_eo_apply_schur_static_status(ctx, 0, MASS, 0, 32, 48) == B.DSLASH_ERR_NULL
        assert B.dslash_eo_apply_schur_static_status(ctx, 2, MASS, 16, 32, 48) == B.DSLASH_ERR_UNSUPPORTED
        assert B.dslash_eo_apply_schur_static_status(ctx, 0, -4.0, 16, 32, 48) == B.DSLASH_ERR_UNSUPPORTED
        assert B.dslash_eo_apply_schur_static_status(ctx, 0, MASS, 24, 32, 48) == B.DSLASH_ERR_ALIGN
        assert B.dslash_eo_apply_schur_static_status(ctx, 0, MASS, 4096, 4096 + 1024, 48) == B.DSLASH_ERR_ALIAS
    finally:
        B.dslash_destroy(ctx)
    ctx = B.dslash_create((3, 4, 4, 4), B.DSLASH_FP64, B.DSLASH_SOA)
    try:
        assert B.dslash_eo_apply_schur_static_status(ctx, 0, MASS, 16, 32, 48) == B.DSLASH_ERR_DIMS
    finally:
        B.dslash_destroy(ctx)

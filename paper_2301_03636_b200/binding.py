"""Thin ctypes binding of libdslash_b200.so: the same names as include/dslash_b200.h, argument
marshalling only.  Every step of the path runs in the library's CUDA kernels; there is no Python or
CPU fallback.  Importing this module loads the library and raises ImportError if it is missing or
does not export a declared symbol (build it with `python -m paper_2301_03636_b200.build`).

Pointers are passed as plain integers (e.g. `tensor.data_ptr()`, `ndarray.ctypes.data`); streams as
the integer value of a cudaStream_t (e.g. `torch.cuda.current_stream().cuda_stream`).  Functions
that return a status in C raise DslashError on a non-zero status here and return their outputs.
"""
import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
# Importing this module always loads the operator library, whatever the environment says.  The measurement build whose kernels
# move the same bytes and compute nothing (python -m paper_2301_03636_b200.build --skeleton) is only ever loaded by an explicit
# load_skeleton() call (bench.py --skeleton makes it); SKELETON is True from then on and results are not the operator.
SKELETON = False
LIB_PATH = os.path.join(_HERE, "libdslash_b200.so")
SKELETON_LIB_PATH = os.path.join(_HERE, "libdslash_b200_skeleton.so")

DSLASH_FP64, DSLASH_FP32 = 0, 1
DSLASH_AOS, DSLASH_SOA, DSLASH_RECON12 = 0, 1, 16
DSLASH_OK = 0
DSLASH_ERR_NULL, DSLASH_ERR_DIMS, DSLASH_ERR_PRECISION, DSLASH_ERR_LAYOUT = -1, -2, -3, -4
DSLASH_ERR_ALIGN, DSLASH_ERR_ALIAS, DSLASH_ERR_UNSUPPORTED, DSLASH_ERR_CUDA, DSLASH_ERR_NOMEM = -5, -6, -7, -8, -9
DSLASH_ERR_TOO_LARGE = -10
DSLASH_STATIC_SCRATCH_BYTES = 8 << 20
DSLASH_VARIANT_TUNED = 0
DSLASH_MAP_MINIMAL, DSLASH_MAP_TOFROM = 0, 1
DSLASH_KERNEL_AUTO, DSLASH_KERNEL_DIRECT = 0, 1
DSLASH_KERNEL_WARP_PIPE, DSLASH_KERNEL_MARCH = 5, 6
MARCH_NW, MARCH_NWS, MARCH_WARP_INTS = 7, 9, 9
MARCH_BLOCK_INTS = 4 + MARCH_NW * MARCH_WARP_INTS  # block plan of dslash_march_plan()
DSLASH_OPT_PIPE_SLOTS, DSLASH_OPT_PIPE_WARPS, DSLASH_OPT_PIPE_ZBLOCK, DSLASH_OPT_TUNE_MODE, DSLASH_OPT_MARCH_LEAD = 7, 8, 9, 10, 11
DSLASH_OPT_MARCH_POLICY = 13
DSLASH_TUNE_BURST, DSLASH_TUNE_SUSTAINED = 0, 1
DSLASH_OPT_OCCUPANCY, DSLASH_OPT_L2_POLICY, DSLASH_OPT_L1_CARVEOUT, DSLASH_OPT_X_SHUFFLE = 2, 3, 4, 5
DSLASH_SCHED_STATIC, DSLASH_SCHED_DYNAMIC, DSLASH_SCHED_GUIDED = 0, 1, 2
DSLASH_OP_D, DSLASH_OP_D_DAGGER, DSLASH_OP_M, DSLASH_OP_M_DAGGER = 0, 1, 2, 3

_c_int_p = ctypes.POINTER(ctypes.c_int)
_c_size_p = ctypes.POINTER(ctypes.c_size_t)
_vp = ctypes.c_void_p

# name -> (restype, argtypes); mirrors include/dslash_b200.h (the operator) and include/dslash_b200_diag.h (dslash_probe_launch,
# dslash_march_stats: measurement aids) one to one
SIGNATURES = {
    "dslash_create": (ctypes.c_int, [ctypes.POINTER(_vp), _c_int_p, ctypes.c_int, ctypes.c_int]),
    "dslash_destroy": (ctypes.c_int, [_vp]),
    "dslash_apply": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp]),
    "dslash_apply_op": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_double, _vp, _vp, _vp, _vp]),
    "dslash_cg_solve": (ctypes.c_int, [_vp, _vp, _vp, _vp, ctypes.c_double, ctypes.c_double, ctypes.c_int, _c_int_p,
                                        ctypes.POINTER(ctypes.c_double), _vp]),
    "dslash_eo_spinor_bytes": (ctypes.c_size_t, [_vp]),
    "dslash_eo_gauge_bytes": (ctypes.c_size_t, [_vp]),
    "dslash_eo_pack_spinor": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int, _vp]),
    "dslash_eo_unpack_spinor": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int, _vp]),
    "dslash_eo_pack_gauge": (ctypes.c_int, [_vp, _vp, _vp, _vp]),
    "dslash_eo_apply": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp, _vp]),
    "dslash_eo_apply_xpay": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp, _vp, ctypes.c_double, ctypes.c_double,
                                             _vp]),
    "dslash_eo_apply_schur": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_double, _vp, _vp, _vp, _vp, _vp]),
    "dslash_static_scratch_bytes": (ctypes.c_size_t, []),
    "dslash_eo_apply_schur_static": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_double, _vp, _vp, _vp, _vp]),
    "dslash_eo_cg_solve": (ctypes.c_int, [_vp, _vp, _vp, _vp, ctypes.c_double, ctypes.c_double, ctypes.c_int, _c_int_p,
                                           ctypes.POINTER(ctypes.c_double), _vp]),
    "dslash_eo_solve": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, _vp, ctypes.c_double, ctypes.c_double, ctypes.c_int, _c_int_p,
                                        ctypes.POINTER(ctypes.c_double), _vp]),
    "dslash_spinor_bytes": (ctypes.c_size_t, [_vp]),
    "dslash_gauge_bytes": (ctypes.c_size_t, [_vp]),
    "dslash_canonical_spinor_bytes": (ctypes.c_size_t, [_vp]),
    "dslash_canonical_gauge_bytes": (ctypes.c_size_t, [_vp]),
    "dslash_pack_spinor": (ctypes.c_int, [_vp, _vp, _vp, _vp]),
    "dslash_unpack_spinor": (ctypes.c_int, [_vp, _vp, _vp, _vp]),
    "dslash_pack_gauge": (ctypes.c_int, [_vp, _vp, _vp, _vp]),
    "dslash_set_variant": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, ctypes.c_int]),
    "dslash_get_variant": (ctypes.c_int, [_vp, _c_int_p, _c_int_p, _c_int_p]),
    "dslash_variant_count": (ctypes.c_int, []),
    "dslash_variant_at": (ctypes.c_int, [ctypes.c_int, _c_int_p, _c_int_p, _c_int_p, _c_int_p]),
    "dslash_omp_variant_count": (ctypes.c_int, [ctypes.c_int]),
    "dslash_omp_variant_at": (ctypes.c_int, [ctypes.c_int, ctypes.c_int, _c_int_p, _c_int_p, _c_int_p, _c_int_p, _c_int_p]),
    "dslash_set_omp_variant": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                               ctypes.c_int]),
    "dslash_set_tile": (ctypes.c_int, [_vp, _c_int_p]),
    "dslash_get_tile": (ctypes.c_int, [_vp, _c_int_p]),
    "dslash_set_time_range": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int]),
    "dslash_get_time_range": (ctypes.c_int, [_vp, _c_int_p, _c_int_p]),
    "dslash_set_kernel": (ctypes.c_int, [_vp, ctypes.c_int]),
    "dslash_get_kernel": (ctypes.c_int, [_vp, _c_int_p]),
    "dslash_slab_face_bytes": (ctypes.c_size_t, [_vp]),
    "dslash_slab_pack_faces": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, _vp]),
    "dslash_slab_interior": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp]),
    "dslash_slab_boundary": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "dslash_march_stats": (ctypes.c_int, [_vp, ctypes.POINTER(ctypes.c_uint), ctypes.c_size_t, _c_int_p]),
    "dslash_march_plan": (ctypes.c_int, [_c_int_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, _c_int_p, ctypes.c_size_t, _c_int_p]),
    "dslash_probe_launch": (ctypes.c_int, [ctypes.c_int, _vp, _vp, ctypes.c_size_t, ctypes.c_int, _vp]),
    "dslash_tune": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, _c_int_p, ctypes.POINTER(ctypes.c_float)]),
    "dslash_set_option": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int]),
    "dslash_get_option": (ctypes.c_int, [_vp, ctypes.c_int, _c_int_p]),
    "dslash_apply_host": (ctypes.c_int, [_vp, _vp, _vp, _vp, ctypes.c_int, _vp, _c_size_p, _c_size_p]),
    "dslash_launch_count": (ctypes.c_longlong, [_vp]),
    "dslash_last_cuda_error": (ctypes.c_int, [_vp]),
    "dslash_error_string": (ctypes.c_char_p, [ctypes.c_int]),
    "dslash_version": (ctypes.c_char_p, []),
}


def _load(path=LIB_PATH, build_hint=""):
    if not os.path.exists(path):
        raise ImportError(
            "%s is missing (%s). Build it: python -m paper_2301_03636_b200.build%s. "
            "There is no CPU fallback." % (os.path.basename(path), path, build_hint))
    try:
        lib = ctypes.CDLL(path)
    except OSError as e:  # pragma: no cover
        raise ImportError("cannot load %s: %s" % (path, e))
    for name, (res, args) in SIGNATURES.items():
        try:
            fn = getattr(lib, name)
        except AttributeError:
            raise ImportError("%s does not export %s" % (path, name))
        fn.restype = res
        fn.argtypes = args
    return lib


_lib = _load()


def load_skeleton() -> None:
    """Measurement aid, for bench.py --skeleton only: route every call of this module to libdslash_b200_skeleton.so, whose
    kernels have their arithmetic compiled out.  From here on nothing this process computes is D psi; SKELETON says so and a
    warning is printed.  Contexts created before the switch belong to the operator library and must not be used after it."""
    global _lib, SKELETON
    import warnings
    _lib = _load(SKELETON_LIB_PATH, " --skeleton")
    SKELETON = True
    warnings.warn("paper_2301_03636_b200.binding now calls the data-movement skeleton: results are NOT the Dslash operator",
                  RuntimeWarning, stacklevel=2)


class DslashError(RuntimeError):
    def __init__(self, status, where):
        self.status = int(status)
        super().__init__("%s: %s" % (where, dslash_error_string(status)))


def _check(status, where):
    if status != DSLASH_OK:
        raise DslashError(status, where)


def _ptr(p):
    return _vp(int(p) if p else None)


def dslash_error_string(status: int) -> str:
    return _lib.dslash_error_string(int(status)).decode()


def dslash_version() -> str:
    return _lib.dslash_version().decode()


def dslash_create(dims, precision: int, layout: int) -> int:
    """Returns the ctx handle (an integer address). dims = (L_X, L_Y, L_Z, L_T)."""
    ctx = _vp()
    arr = (ctypes.c_int * 4)(*[int(d) for d in dims]) if dims is not None else None
    _check(_lib.dslash_create(ctypes.byref(ctx), arr, int(precision), int(layout)), "dslash_create")
    return ctx.value


def dslash_destroy(ctx) -> None:
    _check(_lib.dslash_destroy(_ptr(ctx)), "dslash_destroy")


def dslash_apply(ctx, out, inp, gauge, stream=0) -> None:
    _check(_lib.dslash_apply(_ptr(ctx), _ptr(out), _ptr(inp), _ptr(gauge), _ptr(stream)), "dslash_apply")


def dslash_apply_status(ctx, out, inp, gauge, stream=0) -> int:
    """dslash_apply returning the raw status instead of raising (error-path tests)."""
    return int(_lib.dslash_apply(_ptr(ctx), _ptr(out), _ptr(inp), _ptr(gauge), _ptr(stream)))


def dslash_apply_op(ctx, op: int, mass: float, out, inp, gauge, stream=0) -> None:
    _check(_lib.dslash_apply_op(_ptr(ctx), int(op), float(mass), _ptr(out), _ptr(inp), _ptr(gauge), _ptr(stream)),
           "dslash_apply_op")


def dslash_cg_solve(ctx, x, b, gauge, mass: float, tol: float, max_iter: int, stream=0):
    """Returns (iterations, rel_residual)."""
    it, rel = ctypes.c_int(), ctypes.c_double()
    _check(_lib.dslash_cg_solve(_ptr(ctx), _ptr(x), _ptr(b), _ptr(gauge), float(mass), float(tol), int(max_iter),
                                ctypes.byref(it), ctypes.byref(rel), _ptr(stream)), "dslash_cg_solve")
    return it.value, rel.value


def dslash_eo_spinor_bytes(ctx) -> int:
    return int(_lib.dslash_eo_spinor_bytes(_ptr(ctx)))


def dslash_eo_gauge_bytes(ctx) -> int:
    return int(_lib.dslash_eo_gauge_bytes(_ptr(ctx)))


def dslash_eo_pack_spinor(ctx, dst_half, src_canonical, parity: int, stream=0) -> None:
    _check(_lib.dslash_eo_pack_spinor(_ptr(ctx), _ptr(dst_half), _ptr(src_canonical), int(parity), _ptr(stream)),
           "dslash_eo_pack_spinor")


def dslash_eo_unpack_spinor(ctx, dst_canonical, src_half, parity: int, stream=0) -> None:
    _check(_lib.dslash_eo_unpack_spinor(_ptr(ctx), _ptr(dst_canonical), _ptr(src_half), int(parity), _ptr(stream)),
           "dslash_eo_unpack_spinor")


def dslash_eo_pack_gauge(ctx, dst_eo, src_canonical, stream=0) -> None:
    _check(_lib.dslash_eo_pack_gauge(_ptr(ctx), _ptr(dst_eo), _ptr(src_canonical), _ptr(stream)), "dslash_eo_pack_gauge")


def dslash_eo_apply(ctx, out_parity: int, dagger: int, out, inp, gauge_eo, stream=0) -> None:
    _check(_lib.dslash_eo_apply(_ptr(ctx), int(out_parity), int(dagger), _ptr(out), _ptr(inp), _ptr(gauge_eo), _ptr(stream)),
           "dslash_eo_apply")


def dslash_eo_apply_status(ctx, out_parity: int, dagger: int, out, inp, gauge_eo, stream=0) -> int:
    """dslash_eo_apply returning the raw status instead of raising (error-path tests)."""
    return int(_lib.dslash_eo_apply(_ptr(ctx), int(out_parity), int(dagger), _ptr(out), _ptr(inp), _ptr(gauge_eo), _ptr(stream)))


def dslash_eo_apply_xpay(ctx, out_parity: int, dagger: int, out, inp, gauge_eo, c, a: float, b: float, stream=0) -> None:
    _check(_lib.dslash_eo_apply_xpay(_ptr(ctx), int(out_parity), int(dagger), _ptr(out), _ptr(inp), _ptr(gauge_eo), _ptr(c),
                                     float(a), float(b), _ptr(stream)), "dslash_eo_apply_xpay")


def dslash_eo_apply_schur(ctx, dagger: int, mass: float, out_even, in_even, tmp_odd, gauge_eo, stream=0) -> None:
    _check(_lib.dslash_eo_apply_schur(_ptr(ctx), int(dagger), float(mass), _ptr(out_even), _ptr(in_even), _ptr(tmp_odd),
                                      _ptr(gauge_eo), _ptr(stream)), "dslash_eo_apply_schur")


def dslash_static_scratch_bytes() -> int:
    return int(_lib.dslash_static_scratch_bytes())


def dslash_eo_apply_schur_static(ctx, dagger: int, mass: float, out_even, in_even, gauge_eo, stream=0) -> None:
    """dslash_eo_apply_schur without a scratch argument, for callers that cannot allocate device memory: the intermediate
    lives in an 8 MiB array inside the library (one per GPU, shared by all calls; see include/dslash_b200.h)."""
    _check(_lib.dslash_eo_apply_schur_static(_ptr(ctx), int(dagger), float(mass), _ptr(out_even), _ptr(in_even), _ptr(gauge_eo),
                                             _ptr(stream)), "dslash_eo_apply_schur_static")


def dslash_eo_apply_schur_static_status(ctx, dagger: int, mass: float, out_even, in_even, gauge_eo, stream=0) -> int:
    return int(_lib.dslash_eo_apply_schur_static(_ptr(ctx), int(dagger), float(mass), _ptr(out_even), _ptr(in_even), _ptr(gauge_eo),
                                                 _ptr(stream)))


def dslash_eo_cg_solve(ctx, x_even, b_even, gauge_eo, mass: float, tol: float, max_iter: int, stream=0):
    """Returns (iterations, rel_residual)."""
    it, rel = ctypes.c_int(), ctypes.c_double()
    _check(_lib.dslash_eo_cg_solve(_ptr(ctx), _ptr(x_even), _ptr(b_even), _ptr(gauge_eo), float(mass), float(tol), int(max_iter),
                                   ctypes.byref(it), ctypes.byref(rel), _ptr(stream)), "dslash_eo_cg_solve")
    return it.value, rel.value


def dslash_eo_solve(ctx, x_even, x_odd, b_even, b_odd, gauge_eo, mass: float, tol: float, max_iter: int, stream=0):
    """Returns (iterations, rel_residual)."""
    it, rel = ctypes.c_int(), ctypes.c_double()
    _check(_lib.dslash_eo_solve(_ptr(ctx), _ptr(x_even), _ptr(x_odd), _ptr(b_even), _ptr(b_odd), _ptr(gauge_eo), float(mass),
                                float(tol), int(max_iter), ctypes.byref(it), ctypes.byref(rel), _ptr(stream)), "dslash_eo_solve")
    return it.value, rel.value


def dslash_spinor_bytes(ctx) -> int:
    return int(_lib.dslash_spinor_bytes(_ptr(ctx)))


def dslash_gauge_bytes(ctx) -> int:
    return int(_lib.dslash_gauge_bytes(_ptr(ctx)))


def dslash_canonical_spinor_bytes(ctx) -> int:
    return int(_lib.dslash_canonical_spinor_bytes(_ptr(ctx)))


def dslash_canonical_gauge_bytes(ctx) -> int:
    return int(_lib.dslash_canonical_gauge_bytes(_ptr(ctx)))


def dslash_pack_spinor(ctx, dst_native, src_canonical, stream=0) -> None:
    _check(_lib.dslash_pack_spinor(_ptr(ctx), _ptr(dst_native), _ptr(src_canonical), _ptr(stream)), "dslash_pack_spinor")


def dslash_unpack_spinor(ctx, dst_canonical, src_native, stream=0) -> None:
    _check(_lib.dslash_unpack_spinor(_ptr(ctx), _ptr(dst_canonical), _ptr(src_native), _ptr(stream)),
           "dslash_unpack_spinor")


def dslash_pack_gauge(ctx, dst_native, src_canonical, stream=0) -> None:
    _check(_lib.dslash_pack_gauge(_ptr(ctx), _ptr(dst_native), _ptr(src_canonical), _ptr(stream)), "dslash_pack_gauge")


def dslash_set_variant(ctx, collapse_depth: int, threads_per_block: int = 0, sites_per_thread: int = 0) -> None:
    _check(_lib.dslash_set_variant(_ptr(ctx), int(collapse_depth), int(threads_per_block), int(sites_per_thread)),
           "dslash_set_variant")


def dslash_get_variant(ctx):
    d, b, s = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    _check(_lib.dslash_get_variant(_ptr(ctx), ctypes.byref(d), ctypes.byref(b), ctypes.byref(s)), "dslash_get_variant")
    return d.value, b.value, s.value


def dslash_variant_count() -> int:
    return int(_lib.dslash_variant_count())


def dslash_variant_at(index: int):
    """(collapse_depth, threads_per_block, sites_per_thread, layout) of sweep variant `index`."""
    d, b, s, l = ctypes.c_int(), ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    _check(_lib.dslash_variant_at(int(index), ctypes.byref(d), ctypes.byref(b), ctypes.byref(s), ctypes.byref(l)),
           "dslash_variant_at")
    return d.value, b.value, s.value, l.value


def dslash_omp_variant_count(num_loops: int) -> int:
    return int(_lib.dslash_omp_variant_count(int(num_loops)))


def dslash_omp_variant_at(num_loops: int, index: int):
    """(parallel_position, distribute_collapse, parallel_collapse, schedule, map_mode) of the paper's variant `index`."""
    v = [ctypes.c_int() for _ in range(5)]
    _check(_lib.dslash_omp_variant_at(int(num_loops), int(index), *[ctypes.byref(i) for i in v]), "dslash_omp_variant_at")
    return tuple(i.value for i in v)


def dslash_set_omp_variant(ctx, parallel_position: int, distribute_collapse: int, parallel_collapse: int, schedule: int,
                           num_teams: int = 0, team_size: int = 128) -> None:
    _check(_lib.dslash_set_omp_variant(_ptr(ctx), int(parallel_position), int(distribute_collapse), int(parallel_collapse),
                                       int(schedule), int(num_teams), int(team_size)), "dslash_set_omp_variant")


def dslash_set_tile(ctx, tile) -> None:
    arr = (ctypes.c_int * 4)(*[int(t) for t in tile])
    _check(_lib.dslash_set_tile(_ptr(ctx), arr), "dslash_set_tile")


def dslash_get_tile(ctx):
    arr = (ctypes.c_int * 4)()
    _check(_lib.dslash_get_tile(_ptr(ctx), arr), "dslash_get_tile")
    return tuple(arr)


def dslash_set_time_range(ctx, t_begin: int, t_end: int) -> None:
    _check(_lib.dslash_set_time_range(_ptr(ctx), int(t_begin), int(t_end)), "dslash_set_time_range")


def dslash_get_time_range(ctx):
    a, b = ctypes.c_int(), ctypes.c_int()
    _check(_lib.dslash_get_time_range(_ptr(ctx), ctypes.byref(a), ctypes.byref(b)), "dslash_get_time_range")
    return a.value, b.value


def dslash_set_kernel(ctx, kernel: int) -> None:
    _check(_lib.dslash_set_kernel(_ptr(ctx), int(kernel)), "dslash_set_kernel")


def dslash_tune(ctx, out, inp, gauge, stream=None):
    """Times the eligible kernels on these buffers, keeps the fastest; returns (kernel, ms per application).  Synchronises."""
    k, ms = ctypes.c_int(0), ctypes.c_float(0.0)
    _check(_lib.dslash_tune(_ptr(ctx), _ptr(out), _ptr(inp), _ptr(gauge), _ptr(stream), ctypes.byref(k), ctypes.byref(ms)),
           "dslash_tune")
    return k.value, ms.value


DSLASH_PROBE_READ, DSLASH_PROBE_WRITE, DSLASH_PROBE_COPY, DSLASH_PROBE_READ4_WRITE1, DSLASH_PROBE_DFMA = 0, 1, 2, 3, 4


def dslash_probe_launch(kind: int, dst, src, n: int, blocks: int, stream=None) -> None:
    _check(_lib.dslash_probe_launch(int(kind), _ptr(dst), _ptr(src), int(n), int(blocks), _ptr(stream)), "dslash_probe_launch")


def dslash_tune_status(ctx, out, inp, gauge, stream=None) -> int:
    """dslash_tune returning the raw status instead of raising (error-path tests)."""
    return int(_lib.dslash_tune(_ptr(ctx), _ptr(out), _ptr(inp), _ptr(gauge), _ptr(stream), None, None))


def dslash_get_kernel(ctx) -> int:
    k = ctypes.c_int()
    _check(_lib.dslash_get_kernel(_ptr(ctx), ctypes.byref(k)), "dslash_get_kernel")
    return k.value


def dslash_march_plan(dims, t_begin: int, t_end: int, wave: int):
    """Host-side block plan of DSLASH_KERNEL_MARCH (no device needed): a list of blocks
    {t0, nt, nact, warps: [{row, fwd, wr, rd, bwd}]}."""
    arr = (ctypes.c_int * 4)(*[int(d) for d in dims])
    nb = ctypes.c_int()
    _check(_lib.dslash_march_plan(arr, int(t_begin), int(t_end), int(wave), None, 0, ctypes.byref(nb)), "dslash_march_plan")
    n = nb.value * MARCH_BLOCK_INTS
    buf = (ctypes.c_int * n)()
    _check(_lib.dslash_march_plan(arr, int(t_begin), int(t_end), int(wave), buf, n, ctypes.byref(nb)), "dslash_march_plan")
    blocks = []
    for b in range(nb.value):
        v = buf[b * MARCH_BLOCK_INTS:(b + 1) * MARCH_BLOCK_INTS]
        warps = []
        for w in range(MARCH_NW):
            q = v[4 + MARCH_WARP_INTS * w:4 + MARCH_WARP_INTS * (w + 1)]
            warps.append(dict(row=q[0], fwd=(q[1], q[2]), wr=(q[3], q[4]), rd=(q[5], q[6]), bwd=(q[7], q[8])))
        blocks.append(dict(t0=v[0], nt=v[1], nact=v[2], warps=warps))
    return blocks


def dslash_slab_face_bytes(ctx) -> int:
    return int(_lib.dslash_slab_face_bytes(_ptr(ctx)))


def dslash_slab_pack_faces(ctx, face_down, face_up, inp, gauge, stream=0) -> None:
    _check(_lib.dslash_slab_pack_faces(_ptr(ctx), _ptr(face_down), _ptr(face_up), _ptr(inp), _ptr(gauge), _ptr(stream)),
           "dslash_slab_pack_faces")


def dslash_slab_interior(ctx, out, inp, gauge, stream=0) -> None:
    _check(_lib.dslash_slab_interior(_ptr(ctx), _ptr(out), _ptr(inp), _ptr(gauge), _ptr(stream)), "dslash_slab_interior")


def dslash_slab_boundary(ctx, out, inp, gauge, face_from_below, face_from_above, stream=0) -> None:
    _check(_lib.dslash_slab_boundary(_ptr(ctx), _ptr(out), _ptr(inp), _ptr(gauge), _ptr(face_from_below), _ptr(face_from_above),
                                     _ptr(stream)), "dslash_slab_boundary")


def dslash_march_stats(ctx):
    """[(sm_id, cycles, ns_at_mid_march)] per block of the last DSLASH_KERNEL_MARCH launch of this ctx (synchronises)."""
    nb = ctypes.c_int()
    _check(_lib.dslash_march_stats(_ptr(ctx), None, 0, ctypes.byref(nb)), "dslash_march_stats")
    if nb.value == 0:
        return []
    buf = (ctypes.c_uint * (3 * nb.value))()
    _check(_lib.dslash_march_stats(_ptr(ctx), buf, 3 * nb.value, ctypes.byref(nb)), "dslash_march_stats")
    return [(buf[3 * i], buf[3 * i + 1], buf[3 * i + 2]) for i in range(nb.value)]


def dslash_set_option(ctx, option: int, value: int) -> None:
    _check(_lib.dslash_set_option(_ptr(ctx), int(option), int(value)), "dslash_set_option")


def dslash_get_option(ctx, option: int) -> int:
    v = ctypes.c_int()
    _check(_lib.dslash_get_option(_ptr(ctx), int(option), ctypes.byref(v)), "dslash_get_option")
    return v.value


def dslash_apply_host(ctx, out_host, in_host, gauge_host, map_mode: int = DSLASH_MAP_MINIMAL, stream=0):
    """Returns (h2d_bytes, d2h_bytes)."""
    h2d, d2h = ctypes.c_size_t(), ctypes.c_size_t()
    _check(_lib.dslash_apply_host(_ptr(ctx), _ptr(out_host), _ptr(in_host), _ptr(gauge_host), int(map_mode), _ptr(stream),
                                  ctypes.byref(h2d), ctypes.byref(d2h)), "dslash_apply_host")
    return h2d.value, d2h.value


def dslash_launch_count(ctx) -> int:
    return int(_lib.dslash_launch_count(_ptr(ctx)))


def dslash_last_cuda_error(ctx) -> int:
    return int(_lib.dslash_last_cuda_error(_ptr(ctx)))

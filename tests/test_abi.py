"""CPU-only checks of the C ABI: the library builds, loads, exports every symbol that
include/dslash_b200.h declares, and validates arguments before touching CUDA.  No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "dslash_b200.h")
DIAG_HEADER = os.path.join(ROOT, "include", "dslash_b200_diag.h")  # measurement aids, kept out of the operator's header


@pytest.fixture(scope="module")
def B():
    from paper_2301_03636_b200 import build
    build.build()  # no-op when the in-tree .so is newer than its sources
    from paper_2301_03636_b200 import binding
    return binding


def declared_symbols(header=None):
    if header is None:  # everything the library exports under the dslash_ prefix: operator header + diagnostics header
        return sorted(set(declared_symbols(HEADER)) | set(declared_symbols(DIAG_HEADER)))
    text = open(header).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dslash_[a-z0-9_]+)\s*\(", text)))


def test_measurement_aids_live_in_their_own_header():
    assert declared_symbols(DIAG_HEADER) == ["dslash_march_stats", "dslash_probe_launch"]
    assert not set(declared_symbols(DIAG_HEADER)) & set(declared_symbols(HEADER))
    assert "DSLASH_PROBE_" not in open(HEADER).read().replace("dslash_b200_diag.h", "")


def test_header_declares_the_north_star_calls():
    names = declared_symbols(HEADER)
    for must in ("dslash_create", "dslash_apply", "dslash_destroy", "dslash_pack_spinor", "dslash_unpack_spinor",
                 "dslash_pack_gauge", "dslash_set_variant", "dslash_apply_host"):
        assert must in names


def test_library_exports_every_declared_symbol(B):
    lib = ctypes.CDLL(B.LIB_PATH)
    for name in declared_symbols():
        assert hasattr(lib, name), name
    # and the binding mirrors the header one to one
    assert sorted(B.SIGNATURES) == declared_symbols()
    for name in declared_symbols():
        assert hasattr(B, name), "binding lacks %s" % name


def test_costmodel_header_symbols_are_exported_and_bound(B):
    """include/advisor_costmodel.h: every declared costmodel_* call is exported by the same library and mirrored by
    paper_2301_03636_b200/costmodel.py; the size queries need no device."""
    text = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "advisor_costmodel.h")).read(), flags=re.S)
    names = sorted(set(re.findall(r"\b(costmodel_[a-z0-9_]+)\s*\(", text)))
    assert "costmodel_train" in names and "costmodel_predict" in names and len(names) == 11
    lib = ctypes.CDLL(B.LIB_PATH)
    from paper_2301_03636_b200 import costmodel as C
    assert sorted(C.SIGNATURES) == names
    for name in names:
        assert hasattr(lib, name) and hasattr(C, name), name
    # "with 33 input features, have 66, 132, 66, and 33 neurons"
    assert C.costmodel_weight_count(33) == 33 * 66 + 66 * 132 + 132 * 66 + 66 * 33 + 33
    assert C.costmodel_param_count(33) == C.costmodel_weight_count(33) + 66 + 132 + 66 + 33 + 1
    assert C.costmodel_param_count(0) == 0 and C.costmodel_weight_count(-1) == 0
    assert C.costmodel_train_smem_bytes(33, 16, 8) < C.costmodel_train_smem_bytes(33, 16, 4) <= 232448
    assert C.costmodel_train_smem_bytes(33, 16, 5) == 0 and C.costmodel_train_smem_bytes(33, 65, 8) == 0
    # argument validation precedes CUDA
    assert C.costmodel_train_status(3, 10, 0, 0, 0, 0, 1, 16, 0.01, 30, 0.1, 1e-4, -1, 1, 0, 0, 0, 0) == B.DSLASH_ERR_NULL
    assert C.costmodel_train_status(0, 10, 8, 8, 8, 8, 1, 16, 0.01, 30, 0.1, 1e-4, -1, 1, 0, 8, 0, 0) == B.DSLASH_ERR_DIMS
    assert C.costmodel_train_status(3, 10, 8, 8, 12, 8, 1, 16, 0.01, 30, 0.1, 1e-4, -1, 1, 0, 8, 0, 0) == B.DSLASH_ERR_ALIGN
    assert C.costmodel_train_status(3, 10, 8, 8, 8, 8, 1, 16, 0.01, 30, 0.1, 1e-4, -1, 1, 3, 8, 0, 0) == B.DSLASH_ERR_UNSUPPORTED
    assert C.costmodel_launch_count() == 0


def test_error_strings(B):
    assert B.dslash_error_string(0) == "DSLASH_OK"
    for code in range(-10, 0):
        s = B.dslash_error_string(code)
        assert s.startswith("DSLASH_ERR_") and "?" not in s
    assert "?" in B.dslash_error_string(-99)
    assert B.dslash_version() == "0.1"


def test_argument_validation_precedes_cuda(B):
    with pytest.raises(B.DslashError) as e:
        B.dslash_create(None, B.DSLASH_FP64, B.DSLASH_SOA)
    assert e.value.status == B.DSLASH_ERR_NULL
    for dims, prec, lay, want in [
        ((4, 4, 0, 4), B.DSLASH_FP64, B.DSLASH_SOA, B.DSLASH_ERR_DIMS),
        ((4, 4, -1, 4), B.DSLASH_FP64, B.DSLASH_SOA, B.DSLASH_ERR_DIMS),
        ((128, 128, 128, 64), B.DSLASH_FP64, B.DSLASH_SOA, B.DSLASH_ERR_DIMS),  # 36 V >= 2^31
        ((4, 4, 4, 4), 2, B.DSLASH_SOA, B.DSLASH_ERR_PRECISION),
        ((4, 4, 4, 4), B.DSLASH_FP64, 2, B.DSLASH_ERR_LAYOUT),
        ((4, 4, 4, 4), B.DSLASH_FP64, 32, B.DSLASH_ERR_LAYOUT),
    ]:
        with pytest.raises(B.DslashError) as e:
            B.dslash_create(dims, prec, lay)
        assert e.value.status == want, (dims, prec, lay)
    # NULL ctx paths
    assert B.dslash_spinor_bytes(None) == 0 and B.dslash_gauge_bytes(None) == 0
    assert B.dslash_launch_count(None) == 0
    B.dslash_destroy(None)  # no-op
    assert B.dslash_apply_status(None, 16, 32, 48) == B.DSLASH_ERR_NULL
    with pytest.raises(B.DslashError) as e:
        B.dslash_set_variant(None, 1, 64, 1)
    assert e.value.status == B.DSLASH_ERR_NULL
    assert B.dslash_tune_status(None, 16, 32, 48) == B.DSLASH_ERR_NULL
    for kind, dst, src, n, blocks, want in [(B.DSLASH_PROBE_COPY, 16, 0, 4, 1, B.DSLASH_ERR_NULL), (B.DSLASH_PROBE_COPY, 0, 16, 4, 1, B.DSLASH_ERR_NULL),
                                            (B.DSLASH_PROBE_COPY, 16, 32, 0, 1, B.DSLASH_ERR_DIMS), (B.DSLASH_PROBE_COPY, 16, 32, 4, 0, B.DSLASH_ERR_DIMS),
                                            (B.DSLASH_PROBE_COPY, 16, 40, 4, 1, B.DSLASH_ERR_ALIGN), (9, 16, 32, 4, 1, B.DSLASH_ERR_UNSUPPORTED)]:
        with pytest.raises(B.DslashError) as e:
            B.dslash_probe_launch(kind, dst, src, n, blocks)
        assert e.value.status == want, (kind, dst, src, n, blocks)


def test_variant_enumeration_is_the_120_of_config_5(B):
    n = B.dslash_variant_count()
    assert n == 120
    seen = {B.dslash_variant_at(i) for i in range(n)}
    assert len(seen) == 120
    assert {v[0] for v in seen} == {1, 2, 3, 4}
    assert {v[1] for v in seen} == {64, 128, 256, 512, 1024}
    assert {v[2] for v in seen} == {1, 2, 4}
    assert {v[3] for v in seen} == {B.DSLASH_AOS, B.DSLASH_SOA}
    for bad in (-1, 120):
        with pytest.raises(B.DslashError) as e:
            B.dslash_variant_at(bad)
        assert e.value.status == B.DSLASH_ERR_UNSUPPORTED


def test_omp_variant_space_reproduces_table_1(B):
    """PAPER.md:166-173 (Table 1): 6, 18, 42, 84 variants for 1..4 nested loops (tests/golden/table1_variant_counts.txt)."""
    golden = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "table1_variant_counts.txt")):
        if line.strip() and not line.startswith("#"):
            n, v = line.split()
            golden[int(n)] = int(v)
    assert golden == {1: 6, 2: 18, 3: 42, 4: 84}
    for n, want in golden.items():
        assert B.dslash_omp_variant_count(n) == want
        seen = set()
        for i in range(want):
            x, a, b, sched, mode = B.dslash_omp_variant_at(n, i)
            assert 0 <= x < n and 1 <= b <= n - x  # max collapse of parallel for is NUM - x
            assert (a == 0) if x == 0 else (1 <= a <= x)  # max collapse of teams distribute is x
            assert sched in (B.DSLASH_SCHED_STATIC, B.DSLASH_SCHED_DYNAMIC, B.DSLASH_SCHED_GUIDED)
            assert mode in (B.DSLASH_MAP_MINIMAL, B.DSLASH_MAP_TOFROM)
            seen.add((x, a, b, sched, mode))
        assert len(seen) == want
        for bad in (-1, want):
            with pytest.raises(B.DslashError):
                B.dslash_omp_variant_at(n, bad)
    assert B.dslash_omp_variant_count(0) == 0 and B.dslash_omp_variant_count(5) == 0
    # loop structures alone: 1, 3, 7, 14
    assert [B.dslash_omp_variant_count(n) // 6 for n in (1, 2, 3, 4)] == [1, 3, 7, 14]


def test_environment_cannot_swap_the_operator_library_for_the_skeleton(B):
    """The measurement build (arithmetic compiled out) is reachable through binding.load_skeleton() only: an ambient
    DSLASH_B200_SKELETON=1, which older revisions obeyed at import, must not change what `import binding` loads."""
    import subprocess
    import sys
    env = dict(os.environ, DSLASH_B200_SKELETON="1")
    code = ("from paper_2301_03636_b200 import binding as B; import os; "
            "assert os.path.basename(B.LIB_PATH) == 'libdslash_b200.so' and B.SKELETON is False; "
            "assert B._lib._name == B.LIB_PATH; print('ok')")
    r = subprocess.run([sys.executable, "-c", code], cwd=ROOT, env=env, capture_output=True, text=True)
    assert r.returncode == 0 and r.stdout.strip() == "ok", r.stderr
    assert callable(B.load_skeleton) and B.SKELETON is False


def test_no_cuda_device_is_an_error_not_a_fallback(B):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(B.DslashError) as e:
        B.dslash_create((4, 4, 4, 4), B.DSLASH_FP64, B.DSLASH_SOA)
    assert e.value.status == B.DSLASH_ERR_CUDA


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2301_03636_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "dslash_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2301_03636_b200\b", text, flags=re.M), f

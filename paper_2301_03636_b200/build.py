"""Build libdslash_b200.so for sm_100a, in-tree (paper_2301_03636_b200/libdslash_b200.so).

    python -m paper_2301_03636_b200.build [--force] [--verbose]
    python -m paper_2301_03636_b200.build --skeleton     # libdslash_b200_skeleton.so: every kernel with its arithmetic
                                                         # compiled out (-DDSLASH_NO_MATH, csrc/dslash_site.cuh), a
                                                         # measurement aid for bench.py --skeleton; never loaded by default

nvcc cross-compiles without a GPU.  Each .cu is compiled to an object (in parallel) and linked with
the static CUDA runtime, so the library has no libcudart.so dependency and can be dlopen'ed on a box
without a GPU (the symbol test) as well as on the B200.
"""
import concurrent.futures
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libdslash_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]
# extra compiler flags for measurement builds (e.g. -DDSLASH_F32X2 / -DDSLASH_SCALAR_F32, csrc/dslash_site.cuh); use with --force
FLAGS += os.environ.get("DSLASH_NVCC_EXTRA", "").split()


def _sources():
    return sorted(f for f in os.listdir(CSRC) if f.endswith(".cu"))


def _deps_mtime():
    m = 0.0
    for root in (CSRC, os.path.join(os.path.dirname(HERE), "include")):
        for f in os.listdir(root):
            m = max(m, os.path.getmtime(os.path.join(root, f)))
    return max(m, os.path.getmtime(os.path.abspath(__file__)))


def _compile(src, verbose, objdir=OBJ, extra=()):
    obj = os.path.join(objdir, src[:-3] + ".o")
    cmd = [NVCC] + ARCH + FLAGS + list(extra) + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, src), "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (src, r.stdout, r.stderr))
    return obj, r.stderr


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _deps_mtime():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    srcs = _sources()
    with concurrent.futures.ThreadPoolExecutor(max_workers=min(8, len(srcs))) as ex:
        results = list(ex.map(lambda s: _compile(s, verbose), srcs))
    if verbose:
        for _, log in results:
            sys.stderr.write(log)
    tmp = LIB + ".tmp%d" % os.getpid()
    cmd = [NVCC] + ARCH + ["-shared", "-cudart", "static", "-o", tmp] + [o for o, _ in results]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n%s\n%s" % (r.stdout, r.stderr))
    os.replace(tmp, LIB)
    return LIB


SKELETON_LIB = os.path.join(HERE, "libdslash_b200_skeleton.so")


def build_skeleton(force: bool = False) -> str:
    """The same library with -DDSLASH_NO_MATH: results are not the operator (see csrc/dslash_site.cuh)."""
    if not force and os.path.exists(SKELETON_LIB) and os.path.getmtime(SKELETON_LIB) >= _deps_mtime():
        return SKELETON_LIB
    objdir = os.path.join(HERE, "build_skeleton")
    os.makedirs(objdir, exist_ok=True)
    srcs = _sources()
    with concurrent.futures.ThreadPoolExecutor(max_workers=min(8, len(srcs))) as ex:
        results = list(ex.map(lambda s: _compile(s, False, objdir, ("-DDSLASH_NO_MATH",)), srcs))
    tmp = SKELETON_LIB + ".tmp%d" % os.getpid()
    r = subprocess.run([NVCC] + ARCH + ["-shared", "-cudart", "static", "-o", tmp] + [o for o, _ in results], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n%s\n%s" % (r.stdout, r.stderr))
    os.replace(tmp, SKELETON_LIB)
    return SKELETON_LIB


if __name__ == "__main__":
    if "--skeleton" in sys.argv:
        print(build_skeleton(force="--force" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))

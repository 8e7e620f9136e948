"""The CPU oracle under AddressSanitizer + UndefinedBehaviorSanitizer (SURVEY.md section 4 tier 4, section 5 "Race detection /
sanitizers"; compute-sanitizer for the CUDA side is closed on the GPU pool).

oracle/dslash_oracle.c is rebuilt with -fsanitize=address,undefined -fno-sanitize-recover=all together with a small C driver
that calls oracle_dslash, oracle_dslash_dagger and oracle_dslash_sites on a lattice with all-different extents (every wrap, a
ragged OpenMP split) and on the one-site lattice (every neighbour is the site itself).  The buffers are exact-size heap
allocations, so an index one past either end of psi, gauge or out is reported.  A report or a non-zero exit fails the test.
"""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "dslash_oracle.c")

DRIVER = r"""
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
int oracle_dslash(double *out, const double *psi, const double *gauge, const int dims[4], int nthreads);
int oracle_dslash_dagger(double *out, const double *psi, const double *gauge, const int dims[4], int nthreads);
int oracle_dslash_sites(double *out, const double *psi, const double *gauge, const int dims[4], const int64_t *sites,
                        int64_t nsites, int nthreads);
static double rnd(uint64_t *s) { *s = *s * 6364136223846793005ull + 1442695040888963407ull; return (double)(*s >> 11) / 9007199254740992.0 - 0.5; }
static int run(const int dims[4], int nthreads) {
    const int64_t V = (int64_t)dims[0] * dims[1] * dims[2] * dims[3];
    double *psi = malloc(sizeof(double) * V * 24), *gauge = malloc(sizeof(double) * V * 72);
    double *out = malloc(sizeof(double) * V * 24), *dag = malloc(sizeof(double) * V * 24), *one = malloc(sizeof(double) * V * 24);
    int64_t *sites = malloc(sizeof(int64_t) * V);
    uint64_t s = 2301036360ull + (uint64_t)V;
    for (int64_t i = 0; i < V * 24; ++i) psi[i] = rnd(&s);
    for (int64_t i = 0; i < V * 72; ++i) gauge[i] = rnd(&s);
    for (int64_t i = 0; i < V; ++i) sites[i] = V - 1 - i;
    int rc = oracle_dslash(out, psi, gauge, dims, nthreads);
    rc |= oracle_dslash_dagger(dag, psi, gauge, dims, nthreads);
    rc |= oracle_dslash_sites(one, psi, gauge, dims, sites, V, nthreads);
    rc |= oracle_dslash_sites(one, psi, gauge, dims, sites, 0, nthreads) != 0;          /* empty list */
    sites[0] = V;
    rc |= oracle_dslash_sites(one, psi, gauge, dims, sites, V, nthreads) != -3;         /* out-of-range site is refused */
    sites[0] = V - 1;
    for (int64_t k = 0; k < V && !rc; ++k)                                             /* the site form equals the full form */
        for (int c = 0; c < 24; ++c) rc |= one[k * 24 + c] != out[(V - 1 - k) * 24 + c];
    double sum = 0.0;
    for (int64_t i = 0; i < V * 24; ++i) sum += out[i] * out[i] + dag[i] * dag[i];
    free(psi); free(gauge); free(out); free(dag); free(one); free(sites);
    if (!(sum > 0.0)) rc |= 64;
    return rc;
}
int main(void) {
    const int a[4] = {3, 2, 4, 5}, b[4] = {1, 1, 1, 1}, c[4] = {2, 1, 3, 1};
    int rc = run(a, 3) | run(a, 1) | run(b, 2) | run(c, 0);
    printf("rc=%d\n", rc);
    return rc;
}
"""


@pytest.mark.skipif(shutil.which("gcc") is None, reason="no gcc")
def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    drv = tmp_path / "driver.c"
    drv.write_text(DRIVER)
    exe = tmp_path / "oracle_san"
    flags = ["-O1", "-g", "-std=c99", "-fcx-limited-range", "-fopenmp", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
             "-fno-omit-frame-pointer"]
    build = subprocess.run(["gcc"] + flags + [SRC, str(drv), "-o", str(exe), "-lm"], capture_output=True, text=True)
    if build.returncode != 0 and ("asan" in build.stderr or "ubsan" in build.stderr or "sanitize" in build.stderr):
        pytest.skip("this gcc has no sanitizer runtime: " + build.stderr.strip().splitlines()[-1])
    assert build.returncode == 0, build.stderr
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0:halt_on_error=1", UBSAN_OPTIONS="print_stacktrace=1",
               OMP_NUM_THREADS="4")
    env.pop("LD_PRELOAD", None)
    run = subprocess.run([str(exe)], capture_output=True, text=True, env=env, timeout=300)
    assert run.returncode == 0, (run.stdout, run.stderr)
    assert run.stdout.strip() == "rc=0"
    assert "ERROR" not in run.stderr and "runtime error" not in run.stderr, run.stderr

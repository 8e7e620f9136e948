/*
 * dslash_oracle.c -- CPU ORACLE for the Wilson Dslash operator.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the plain, slow, obviously-correct restatement of the operator the CUDA library
 * computes.  It exists to be compared against; it is NOT part of the product path.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or
 * call it.  It shares no code, header, table or helper with paper_2301_03636_b200/csrc (the gamma
 * matrices below are typed out here a second time on purpose).
 *
 * What it computes (section 1.1, Eq. 1, read as DESIGN.md "Readings" R1-R8):
 *
 *   out(x)[a][i] = sum_{mu=0..3} sum_{b=0..3} sum_{j=0..2}
 *        [ (1 - gamma_mu)[a][b] * U_mu(x)[i][j]            * psi(x+mu^)[b][j]
 *        + (1 + gamma_mu)[a][b] * conj( U_mu(x-mu^)[j][i] ) * psi(x-mu^)[b][j] ]
 *
 *   - x +- mu^ are taken modulo L_mu ("periodic lattice"; the Kronecker deltas of Eq. 1).
 *   - Eq. 1 as printed has U^dagger_mu(x+mu^) in the backward term; that is a typo (it breaks gauge
 *     covariance, tests/test_oracle_pins.py::test_gauge_covariance).  BASELINE.json's north_star
 *     states the operator with U^dagger_mu(x-mu^), which is what is written here.  (Reading R1)
 *   - No 1/2, no mass term, no overall sign: Eq. 1 has none.  (Reading R3)
 *   - gamma_mu: the paper only says "4x4 Dirac matrices that are fixed"; BASELINE.json
 *     configs[0] fixes the DeGrand-Rossi basis.  The matrices are typed out below.  (Reading R4)
 *   - mu = 0,1,2,3 <-> x,y,z,t (Eq. 1 writes mu = 1..4).  (Reading R5)
 *   - Fields are flat arrays: site index s = x + L_X*(y + L_Y*(z + L_Z*t)), i.e. the
 *     four loops of Code 1 run t,z,y,x outer->inner and x is
 *     memory-fastest.  Spinor real index ((s*4 + a)*3 + c)*2 + ri  (ri 0 = re, 1 = im);
 *     gauge real index (((s*4 + mu)*3 + i)*3 + j)*2 + ri, row-major, (U v)[i] = sum_j U[i][j] v[j].
 *     (Readings R6, R7)
 *   - Precision: fp64 (double _Complex) throughout.  (Reading R9)
 *
 * No spin projection, no link compression, no blocking, no reordering: the full 4x4 gamma
 * multiplication is carried out as written.  Summation order: mu ascending, forward term then
 * backward term, b then j innermost.
 *
 * Pins (tests/test_oracle_pins.py): P1 constant spinor, P2 plane wave on an all-different-extent
 * lattice, P3 FFT of a random free field, P4 constant diagonal links, P5 gamma5-hermiticity of the
 * brute-force dense matrix on 2^4, P6 gauge covariance, P7 dense Kronecker-delta matrix built in
 * NumPy straight from Eq. 1, P8 translation covariance, P9 even/odd parity, P10 norm bound and
 * linearity, P11 second moment.  Every exported function below is pinned by these.
 *
 * Build: gcc -O2 -std=c99 -fcx-limited-range -fopenmp -fPIC -shared (see oracle/build.py; the flag makes
 * a complex product the four-multiply textbook formula instead of a call to __muldc3).  OpenMP is used only to
 * split the outermost (t) loop across cores when the oracle is timed as the CPU baseline.
 */
#include <complex.h>
#include <stddef.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double _Complex cplx;

#define NS 4 /* SPINS */
#define NC 3 /* COLORS */

/* DeGrand-Rossi gamma matrices, gamma_mu[a][b], mu = 0(x),1(y),2(z),3(t).  Entries are
 * {re, im} pairs so that the table is plain data.  (DESIGN.md Reading R4.)
 *
 *  g0 = [ 0  0  0  i ]  g1 = [ 0  0  0 -1 ]  g2 = [ 0  0  i  0 ]  g3 = [ 0  0  1  0 ]
 *       [ 0  0  i  0 ]       [ 0  0  1  0 ]       [ 0  0  0 -i ]       [ 0  0  0  1 ]
 *       [ 0 -i  0  0 ]       [ 0  1  0  0 ]       [-i  0  0  0 ]       [ 1  0  0  0 ]
 *       [-i  0  0  0 ]       [-1  0  0  0 ]       [ 0  i  0  0 ]       [ 0  1  0  0 ]
 */
static const double GAMMA[4][NS][NS][2] = {
    /* gamma_0 (x) */
    {{{0, 0}, {0, 0}, {0, 0}, {0, 1}},
     {{0, 0}, {0, 0}, {0, 1}, {0, 0}},
     {{0, 0}, {0, -1}, {0, 0}, {0, 0}},
     {{0, -1}, {0, 0}, {0, 0}, {0, 0}}},
    /* gamma_1 (y) */
    {{{0, 0}, {0, 0}, {0, 0}, {-1, 0}},
     {{0, 0}, {0, 0}, {1, 0}, {0, 0}},
     {{0, 0}, {1, 0}, {0, 0}, {0, 0}},
     {{-1, 0}, {0, 0}, {0, 0}, {0, 0}}},
    /* gamma_2 (z) */
    {{{0, 0}, {0, 0}, {0, 1}, {0, 0}},
     {{0, 0}, {0, 0}, {0, 0}, {0, -1}},
     {{0, -1}, {0, 0}, {0, 0}, {0, 0}},
     {{0, 0}, {0, 1}, {0, 0}, {0, 0}}},
    /* gamma_3 (t) */
    {{{0, 0}, {0, 0}, {1, 0}, {0, 0}},
     {{0, 0}, {0, 0}, {0, 0}, {1, 0}},
     {{1, 0}, {0, 0}, {0, 0}, {0, 0}},
     {{0, 0}, {1, 0}, {0, 0}, {0, 0}}},
};

static cplx gamma_entry(int mu, int a, int b) {
    return GAMMA[mu][a][b][0] + GAMMA[mu][a][b][1] * I;
}

/* Copy gamma_mu into out[4][4][2] (re, im) so that the tests can check the Clifford algebra and
 * the basis against their own typed-out copy. */
void oracle_gamma(int mu, double *out) {
    for (int a = 0; a < NS; ++a)
        for (int b = 0; b < NS; ++b) {
            out[(a * NS + b) * 2 + 0] = GAMMA[mu][a][b][0];
            out[(a * NS + b) * 2 + 1] = GAMMA[mu][a][b][1];
        }
}

static size_t site_index(const int dims[4], const int c[4]) {
    /* s = x + L_X*(y + L_Y*(z + L_Z*t))  (Reading R6) */
    return (size_t)c[0] +
           (size_t)dims[0] * ((size_t)c[1] + (size_t)dims[1] * ((size_t)c[2] + (size_t)dims[2] * (size_t)c[3]));
}

static cplx spinor_at(const double *psi, size_t s, int a, int c) {
    const double *p = psi + ((s * NS + (size_t)a) * NC + (size_t)c) * 2;
    return p[0] + p[1] * I;
}

static cplx link_at(const double *gauge, size_t s, int mu, int i, int j) {
    const double *p = gauge + (((s * 4 + (size_t)mu) * NC + (size_t)i) * NC + (size_t)j) * 2;
    return p[0] + p[1] * I;
}

/* out24 <- (D psi)(x) (sigma = +1) or (D^dagger psi)(x) (sigma = -1) for the one site with coordinates
 * coord = {x,y,z,t}.  Eq. 1 term by term.  The adjoint of Eq. 1 follows from gamma_mu^dagger = gamma_mu and
 * (U_mu(x) delta_{x+mu,y})^dagger = U_mu(x)^dagger delta_{x,y+mu}: relabelling, D^dagger is Eq. 1 with
 * gamma_mu -> -gamma_mu, i.e. the projectors (1 - sigma*gamma_mu) forward and (1 + sigma*gamma_mu) backward
 * (DESIGN.md Reading R19; pinned by <phi, D psi> = <D^dagger phi, psi> and by gamma_5 D gamma_5 = D^dagger). */
static void dslash_one_site(double *out24, const double *psi, const double *gauge, const int dims[4],
                            const int coord[4], double sigma) {
    cplx acc[NS][NC];
    for (int a = 0; a < NS; ++a)
        for (int i = 0; i < NC; ++i) acc[a][i] = 0.0;

    const size_t s = site_index(dims, coord);

    for (int mu = 0; mu < 4; ++mu) {
        int fwd[4] = {coord[0], coord[1], coord[2], coord[3]};
        int bwd[4] = {coord[0], coord[1], coord[2], coord[3]};
        fwd[mu] = (coord[mu] + 1) % dims[mu];            /* delta_{x+mu^, y} */
        bwd[mu] = (coord[mu] - 1 + dims[mu]) % dims[mu]; /* delta_{x-mu^, y} */
        const size_t sf = site_index(dims, fwd);
        const size_t sb = site_index(dims, bwd);

        /* forward:  (1 - sigma*gamma_mu)[a][b] U_mu(x)[i][j] psi(x+mu^)[b][j] */
        for (int a = 0; a < NS; ++a)
            for (int i = 0; i < NC; ++i)
                for (int b = 0; b < NS; ++b) {
                    const cplx pm = (a == b ? 1.0 : 0.0) - sigma * gamma_entry(mu, a, b);
                    for (int j = 0; j < NC; ++j) acc[a][i] += pm * link_at(gauge, s, mu, i, j) * spinor_at(psi, sf, b, j);
                }

        /* backward: (1 + sigma*gamma_mu)[a][b] conj(U_mu(x-mu^)[j][i]) psi(x-mu^)[b][j] */
        for (int a = 0; a < NS; ++a)
            for (int i = 0; i < NC; ++i)
                for (int b = 0; b < NS; ++b) {
                    const cplx pp = (a == b ? 1.0 : 0.0) + sigma * gamma_entry(mu, a, b);
                    for (int j = 0; j < NC; ++j)
                        acc[a][i] += pp * conj(link_at(gauge, sb, mu, j, i)) * spinor_at(psi, sb, b, j);
                }
    }

    for (int a = 0; a < NS; ++a)
        for (int i = 0; i < NC; ++i) {
            out24[(a * NC + i) * 2 + 0] = creal(acc[a][i]);
            out24[(a * NC + i) * 2 + 1] = cimag(acc[a][i]);
        }
}

/* out <- D[gauge] psi on the whole lattice.  dims = {L_X, L_Y, L_Z, L_T}, each >= 1.
 * Four explicit loops t,z,y,x as in Code 1.  nthreads <= 0: all cores. */
static int dslash_all(double *out, const double *psi, const double *gauge, const int dims[4], int nthreads, double sigma) {
    if (!out || !psi || !gauge || !dims) return -1;
    for (int d = 0; d < 4; ++d)
        if (dims[d] < 1) return -2;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
    (void)nthreads;
#pragma omp parallel for num_threads(nthreads) schedule(static)
    for (int t = 0; t < dims[3]; ++t)
        for (int z = 0; z < dims[2]; ++z)
            for (int y = 0; y < dims[1]; ++y)
                for (int x = 0; x < dims[0]; ++x) {
                    const int coord[4] = {x, y, z, t};
                    const size_t s = site_index(dims, coord);
                    dslash_one_site(out + s * (NS * NC * 2), psi, gauge, dims, coord, sigma);
                }
    return 0;
}

int oracle_dslash(double *out, const double *psi, const double *gauge, const int dims[4], int nthreads) {
    return dslash_all(out, psi, gauge, dims, nthreads, 1.0);
}

/* out <- D^dagger[gauge] psi on the whole lattice (see dslash_one_site). */
int oracle_dslash_dagger(double *out, const double *psi, const double *gauge, const int dims[4], int nthreads) {
    return dslash_all(out, psi, gauge, dims, nthreads, -1.0);
}

/* out[n][24] <- (D psi)(sites[k]) for a list of linear site indices: the "one by one" form used
 * for sampled parity at lattice sizes where a full oracle apply is not wanted. */
int oracle_dslash_sites(double *out, const double *psi, const double *gauge, const int dims[4],
                        const int64_t *sites, int64_t nsites, int nthreads) {
    if (!out || !psi || !gauge || !dims || (!sites && nsites > 0)) return -1;
    for (int d = 0; d < 4; ++d)
        if (dims[d] < 1) return -2;
    const int64_t V = (int64_t)dims[0] * dims[1] * dims[2] * dims[3];
    for (int64_t k = 0; k < nsites; ++k)
        if (sites[k] < 0 || sites[k] >= V) return -3;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
    (void)nthreads;
#pragma omp parallel for num_threads(nthreads) schedule(static)
    for (int64_t k = 0; k < nsites; ++k) {
        int64_t r = sites[k];
        int coord[4];
        coord[0] = (int)(r % dims[0]); r /= dims[0];
        coord[1] = (int)(r % dims[1]); r /= dims[1];
        coord[2] = (int)(r % dims[2]); r /= dims[2];
        coord[3] = (int)r;
        dslash_one_site(out + k * (NS * NC * 2), psi, gauge, dims, coord, 1.0);
    }
    return 0;
}

/* Number of threads a call with nthreads <= 0 would use (reported as cpu_baseline.cores). */
int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

"""Pins for the CPU oracle (oracle/dslash_oracle.c): it is checked against what Eq. 1
and the mathematics fix, never against itself and never against the CUDA path.

The paper prints no worked numerical example of D psi, so there is no golden value file for the
operator; every pin below is a closed form, an invariant, a library routine (FFT) or brute force
from the Kronecker-delta form of Eq. 1 written independently here in NumPy.  The gamma matrices
are typed out in this file a second time (from DESIGN.md Reading R4) so that a typo in either copy
fails.  P-numbers follow DESIGN.md "Oracle pins".
"""
import itertools

import numpy as np
import pytest

import oracle
from paper_2301_03636_b200 import inputs

I = 1j
# DeGrand-Rossi basis, DESIGN.md Reading R4 (typed independently of oracle/dslash_oracle.c).
G = np.zeros((4, 4, 4), dtype=np.complex128)
G[0] = [[0, 0, 0, I], [0, 0, I, 0], [0, -I, 0, 0], [-I, 0, 0, 0]]
G[1] = [[0, 0, 0, -1], [0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, 0]]
G[2] = [[0, 0, I, 0], [0, 0, 0, -I], [-I, 0, 0, 0], [0, I, 0, 0]]
G[3] = [[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]]
G5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(np.complex128)
ID4 = np.eye(4, dtype=np.complex128)

DISTINCT = (4, 6, 8, 10)  # (L_X, L_Y, L_Z, L_T), all different, all even


# ------------------------------------------------------------------ helpers (layout only)
def c2r(a):
    """complex [...] -> float64 [..., 2]"""
    return np.ascontiguousarray(np.stack([a.real, a.imag], axis=-1))


def r2c(a):
    return a[..., 0] + 1j * a[..., 1]


def shape4(dims):
    lx, ly, lz, lt = dims
    return (lt, lz, ly, lx)


def unit_gauge(dims):
    u = np.zeros(shape4(dims) + (4, 3, 3), dtype=np.complex128)
    u[..., :, range(3), range(3)] = 1.0
    return u


def random_spinor(dims, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(shape4(dims) + (4, 3)) + 1j * rng.standard_normal(shape4(dims) + (4, 3))


def random_gauge(dims, seed):
    return r2c(inputs.gauge_field(dims, seed))


def apply(u, psi, dims):
    return r2c(oracle.dslash(c2r(psi), c2r(u), dims))


def coords(dims):
    """integer coordinate grids x, y, z, t of shape [T, Z, Y, X]"""
    lx, ly, lz, lt = dims
    t, z, y, x = np.meshgrid(np.arange(lt), np.arange(lz), np.arange(ly), np.arange(lx), indexing="ij")
    return x, y, z, t


def free_matrix(p):
    """M(p) = 2 sum_mu cos p_mu - 2i sum_mu gamma_mu sin p_mu: what Eq. 1 does to e^{ipx} at U = 1:
    (1-g) e^{ip} + (1+g) e^{-ip} = 2 cos p - 2i g sin p."""
    m = np.zeros((4, 4), dtype=np.complex128)
    for mu in range(4):
        m += 2.0 * np.cos(p[mu]) * ID4 - 2j * np.sin(p[mu]) * G[mu]
    return m


def dense_from_eq1(u, dims, gam=G, printed_typo=False):
    """Brute-force dense matrix straight from the Kronecker-delta form of Eq. 1 (P7), independent of
    the oracle's apply routine.  Row/column index = s*12 + spin*3 + colour.
    printed_typo=True builds the equation exactly as printed (backward link taken at x+mu)."""
    lx, ly, lz, lt = dims
    ext = (lx, ly, lz, lt)
    v = lx * ly * lz * lt
    d = np.zeros((v * 12, v * 12), dtype=np.complex128)

    def sidx(c):
        return c[0] + lx * (c[1] + ly * (c[2] + lz * c[3]))

    for c in itertools.product(range(lx), range(ly), range(lz), range(lt)):
        c = list(c)
        s = sidx(c)
        for mu in range(4):
            f = list(c)
            f[mu] = (c[mu] + 1) % ext[mu]
            b = list(c)
            b[mu] = (c[mu] - 1) % ext[mu]
            sf, sb = sidx(f), sidx(b)
            u_x = u[c[3], c[2], c[1], c[0], mu]
            lb = f if printed_typo else b
            u_b = u[lb[3], lb[2], lb[1], lb[0], mu]
            d[s * 12:(s + 1) * 12, sf * 12:(sf + 1) * 12] += np.kron(ID4 - gam[mu], u_x)
            d[s * 12:(s + 1) * 12, sb * 12:(sb + 1) * 12] += np.kron(ID4 + gam[mu], u_b.conj().T)
    return d


def dense_from_oracle(u, dims):
    """Dense matrix of the oracle: column k = D e_k."""
    v = int(np.prod(dims))
    n = v * 12
    cols = np.zeros((n, n), dtype=np.complex128)
    for k in range(n):
        e = np.zeros(n, dtype=np.complex128)
        e[k] = 1.0
        cols[:, k] = apply(u, e.reshape(shape4(dims) + (4, 3)), dims).reshape(n)
    return cols


# ------------------------------------------------------------------ gamma basis
def test_gamma_table_matches_and_clifford():
    for mu in range(4):
        g = oracle.gamma(mu)
        assert np.array_equal(g, G[mu])
        assert np.array_equal(g.conj().T, g)  # hermitian
    for mu in range(4):
        for nu in range(4):
            anti = oracle.gamma(mu) @ oracle.gamma(nu) + oracle.gamma(nu) @ oracle.gamma(mu)
            assert np.array_equal(anti, 2.0 * (mu == nu) * ID4)
    g5 = oracle.gamma(0) @ oracle.gamma(1) @ oracle.gamma(2) @ oracle.gamma(3)
    assert np.array_equal(g5, G5)


# ------------------------------------------------------------------ P1
def test_p1_unit_gauge_constant_spinor_gives_8psi():
    dims = DISTINCT
    chi = np.random.default_rng(1).standard_normal((4, 3)) + 1j * np.random.default_rng(2).standard_normal((4, 3))
    psi = np.broadcast_to(chi, shape4(dims) + (4, 3)).copy()
    out = apply(unit_gauge(dims), psi, dims)
    assert np.abs(out - 8.0 * psi).max() < 1e-13


# ------------------------------------------------------------------ P2
@pytest.mark.parametrize("n", [(1, 2, 3, 4), (3, 1, 5, 7), (0, 5, 2, 9)])
def test_p2_plane_wave_free_wilson(n):
    dims = DISTINCT
    p = [2.0 * np.pi * n[mu] / dims[mu] for mu in range(4)]
    x, y, z, t = coords(dims)
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    rng = np.random.default_rng(7)
    chi = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    psi = phase[..., None, None] * chi
    out = apply(unit_gauge(dims), psi, dims)
    m = free_matrix(p)
    want = phase[..., None, None] * (m @ chi)
    assert np.abs(out - want).max() < 2e-13
    # analytic free-Wilson eigenvalues: 2 sum cos p +- 2i sqrt(sum sin^2 p), each twice
    ev = np.linalg.eigvals(m)
    c = 2.0 * sum(np.cos(p))
    s = 2.0 * np.sqrt(sum(np.sin(q) ** 2 for q in p))
    assert np.allclose(ev.real, c, atol=1e-12)
    assert np.allclose(np.sort(ev.imag), [-s, -s, s, s], atol=1e-12)
    # and the oracle output is an eigen-combination: projecting onto an eigenvector of M(p)
    w, vecs = np.linalg.eig(m)
    chi_e = vecs[:, [0]] * np.array([[1.0, 0.5 - 0.25j, -2.0]])  # eigen-spinor x arbitrary colour
    out_e = apply(unit_gauge(dims), phase[..., None, None] * chi_e, dims)
    assert np.abs(out_e - w[0] * phase[..., None, None] * chi_e).max() < 2e-13


# ------------------------------------------------------------------ P3
def test_p3_free_field_equals_fft_multiplier():
    dims = DISTINCT
    lx, ly, lz, lt = dims
    psi = random_spinor(dims, 11)
    out = apply(unit_gauge(dims), psi, dims)
    pt, pz, py, px = np.meshgrid(*(2.0 * np.pi * np.fft.fftfreq(n) for n in (lt, lz, ly, lx)), indexing="ij")
    m = np.zeros(shape4(dims) + (4, 4), dtype=np.complex128)
    for mu, p in enumerate((px, py, pz, pt)):
        m += 2.0 * np.cos(p)[..., None, None] * ID4 - 2j * np.sin(p)[..., None, None] * G[mu]
    ft = np.fft.fftn(psi, axes=(0, 1, 2, 3))
    want = np.fft.ifftn(np.einsum("tzyxab,tzyxbc->tzyxac", m, ft), axes=(0, 1, 2, 3))
    assert np.abs(out - want).max() < 5e-13


# ------------------------------------------------------------------ P4
def test_p4_constant_diagonal_links_shift_momentum_per_colour():
    dims = DISTINCT
    rng = np.random.default_rng(5)
    theta = rng.uniform(-np.pi, np.pi, size=(4, 3))
    theta[:, 2] = -(theta[:, 0] + theta[:, 1])  # det = 1
    u = np.zeros(shape4(dims) + (4, 3, 3), dtype=np.complex128)
    for mu in range(4):
        for c in range(3):
            u[..., mu, c, c] = np.exp(1j * theta[mu, c])
    n = (1, 2, 3, 4)
    p = np.array([2.0 * np.pi * n[mu] / dims[mu] for mu in range(4)])
    x, y, z, t = coords(dims)
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    chi = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    out = apply(u, phase[..., None, None] * chi, dims)
    want = np.empty_like(out)
    for c in range(3):
        want[..., c] = phase[..., None] * (free_matrix(p + theta[:, c]) @ chi[:, c])
    assert np.abs(out - want).max() < 2e-13
    # the U <-> U^dagger swap must NOT pass (this is what P4 is for)
    swapped = np.empty_like(out)
    for c in range(3):
        swapped[..., c] = phase[..., None] * (free_matrix(p - theta[:, c]) @ chi[:, c])
    assert np.abs(out - swapped).max() > 1.0


# ------------------------------------------------------------------ P5 + P7
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (3, 2, 4, 2)])
def test_p7_dense_kronecker_matrix_equals_oracle(dims):
    u = random_gauge(dims, 21)
    d_eq1 = dense_from_eq1(u, dims)
    psi = random_spinor(dims, 22)
    want = (d_eq1 @ psi.reshape(-1)).reshape(psi.shape)
    out = apply(u, psi, dims)
    assert np.abs(out - want).max() < 1e-13


def test_p5_gamma5_hermiticity_dense_2x2x2x2():
    dims = (2, 2, 2, 2)
    u = random_gauge(dims, 31)
    d = dense_from_oracle(u, dims)  # 192 x 192, column by column through the oracle
    assert d.shape == (192, 192)
    g5 = np.kron(np.eye(16), np.kron(G5, np.eye(3)))
    assert np.abs(g5 @ d @ g5 - d.conj().T).max() < 1e-14
    # the same matrix from the Kronecker-delta form; and D^dagger = D with gamma -> -gamma
    assert np.abs(d - dense_from_eq1(u, dims)).max() < 1e-14
    assert np.abs(d.conj().T - dense_from_eq1(u, dims, gam=-G)).max() < 1e-14


def test_dagger_is_the_adjoint_and_gamma5_conjugate():
    """oracle_dslash_dagger (Reading R19): <phi, D psi> = <D^dagger phi, psi>; D^dagger = gamma5 D gamma5; and on the
    dense 2^4 matrix D^dagger is the conjugate transpose."""
    dims = DISTINCT
    u = random_gauge(dims, 33)
    psi, phi = random_spinor(dims, 34), random_spinor(dims, 35)
    d_psi = apply(u, psi, dims)
    dd_phi = r2c(oracle.dslash_dagger(c2r(phi), c2r(u), dims))
    lhs = np.vdot(phi, d_psi)
    rhs = np.vdot(dd_phi, psi)
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)
    g5 = np.array([1.0, 1.0, -1.0, -1.0])[:, None]
    assert np.abs(dd_phi - g5 * apply(u, g5 * phi, dims)).max() < 2e-13
    small = (2, 2, 2, 2)
    us = random_gauge(small, 36)
    n = 16 * 12
    cols = np.zeros((n, n), dtype=np.complex128)
    for k in range(n):
        e = np.zeros(n, dtype=np.complex128)
        e[k] = 1.0
        cols[:, k] = r2c(oracle.dslash_dagger(c2r(e.reshape(shape4(small) + (4, 3))), c2r(us), small)).reshape(n)
    assert np.abs(cols - dense_from_eq1(us, small).conj().T).max() < 1e-14


def test_wilson_matrix_definition_and_normal_operator_is_positive():
    dims = (4, 2, 6, 4)
    u = random_gauge(dims, 37)
    psi = random_spinor(dims, 38)
    m = 0.1
    mp = r2c(oracle.wilson(c2r(psi), c2r(u), dims, m))
    assert np.abs(mp - ((4.0 + m) * psi - 0.5 * apply(u, psi, dims))).max() < 1e-14
    # free field: M e^{ipx} chi = [(4 + m) - sum cos p + i sum gamma sin p] e^{ipx} chi
    n = (1, 0, 2, 3)
    p = [2.0 * np.pi * n[k] / dims[k] for k in range(4)]
    x, y, z, t = coords(dims)
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    chi = np.random.default_rng(3).standard_normal((4, 3)) + 0j
    got = r2c(oracle.wilson(c2r(phase[..., None, None] * chi), c2r(unit_gauge(dims)), dims, m))
    mm = (4.0 + m) * ID4 - 0.5 * free_matrix(p)
    assert np.abs(got - phase[..., None, None] * (mm @ chi)).max() < 2e-13
    # <psi, M^dagger M psi> = |M psi|^2 > 0
    mdm = r2c(oracle.wilson(c2r(mp), c2r(u), dims, m, dagger=True))
    assert abs(np.vdot(psi, mdm) - np.vdot(mp, mp)) <= 1e-12 * abs(np.vdot(mp, mp))


# ------------------------------------------------------------------ P6
def _gauge_transform(u, psi, g, dims):
    ug = np.empty_like(u)
    for mu in range(4):
        g_fwd = np.roll(g, -1, axis=3 - mu)  # G(x + mu^)
        ug[..., mu, :, :] = g @ u[..., mu, :, :] @ np.conj(np.swapaxes(g_fwd, -1, -2))
    psig = np.einsum("tzyxij,tzyxaj->tzyxai", g, psi)
    return ug, psig


def test_p6_gauge_covariance():
    dims = DISTINCT
    v = int(np.prod(dims))
    u = random_gauge(dims, 41)
    psi = random_spinor(dims, 42)
    g = inputs.haar_su3(v, np.random.default_rng(43)).reshape(shape4(dims) + (3, 3))
    ug, psig = _gauge_transform(u, psi, g, dims)
    lhs = apply(ug, psig, dims)
    rhs = np.einsum("tzyxij,tzyxaj->tzyxai", g, apply(u, psi, dims))
    assert np.abs(lhs - rhs).max() < 2e-13


def test_p6_detects_the_printed_typo_in_eq1():
    """Reading R1: Eq. 1 as printed (backward link at x+mu) is NOT gauge covariant; the corrected
    form is.  Shown on the dense matrices so the oracle is not involved in its own justification."""
    dims = (3, 2, 4, 2)
    v = int(np.prod(dims))
    u = random_gauge(dims, 51)
    psi = random_spinor(dims, 52)
    g = inputs.haar_su3(v, np.random.default_rng(53)).reshape(shape4(dims) + (3, 3))
    ug, psig = _gauge_transform(u, psi, g, dims)

    def cov_err(typo):
        lhs = (dense_from_eq1(ug, dims, printed_typo=typo) @ psig.reshape(-1)).reshape(psi.shape)
        rhs = (dense_from_eq1(u, dims, printed_typo=typo) @ psi.reshape(-1)).reshape(psi.shape)
        return np.abs(lhs - np.einsum("tzyxij,tzyxaj->tzyxai", g, rhs)).max()

    assert cov_err(False) < 1e-13
    assert cov_err(True) > 1.0


# ------------------------------------------------------------------ P8
@pytest.mark.parametrize("mu", [0, 1, 2, 3])
def test_p8_translation_covariance_is_exact(mu):
    dims = (4, 6, 2, 3)
    u = random_gauge(dims, 61)
    psi = random_spinor(dims, 62)
    out = apply(u, psi, dims)
    ax = 3 - mu
    out_r = apply(np.roll(u, 1, axis=ax), np.roll(psi, 1, axis=ax), dims)
    assert np.array_equal(out_r, np.roll(out, 1, axis=ax))


# ------------------------------------------------------------------ P9
def test_p9_even_sites_map_to_odd_sites():
    dims = DISTINCT
    u = random_gauge(dims, 71)
    psi = random_spinor(dims, 72)
    x, y, z, t = coords(dims)
    even = ((x + y + z + t) % 2 == 0)
    psi[~even] = 0.0
    out = apply(u, psi, dims)
    assert np.all(out[even] == 0.0)
    assert np.abs(out[~even]).min() > 0.0


# ------------------------------------------------------------------ P10
def test_p10_norm_bound_and_linearity():
    dims = (4, 2, 6, 4)
    u = random_gauge(dims, 81)
    psi, phi = random_spinor(dims, 82), random_spinor(dims, 83)
    a, b = 0.3 - 1.7j, -2.2 + 0.4j
    lhs = apply(u, a * psi + b * phi, dims)
    rhs = a * apply(u, psi, dims) + b * apply(u, phi, dims)
    assert np.abs(lhs - rhs).max() < 2e-13
    assert np.linalg.norm(apply(u, psi, dims)) <= 8.0 * np.linalg.norm(psi)


# ------------------------------------------------------------------ P11
def test_p11_second_moment_is_32():
    dims = (8, 8, 8, 8)
    gauge, psi = inputs.fields(dims, inputs.BASE_SEED + 99)
    out = r2c(oracle.dslash(psi, gauge, dims))
    m2 = np.mean(np.abs(out) ** 2)
    assert abs(m2 - 32.0) < 0.5  # 49152 components: sigma ~ 32*sqrt(2/49152)*O(few) ~ 0.3


# ------------------------------------------------------------------ sampled form == full form
def test_sites_form_is_the_same_arithmetic():
    dims = (4, 6, 2, 3)
    gauge, psi = inputs.fields(dims, 5)
    full = oracle.dslash(psi, gauge, dims).reshape(-1, 4, 3, 2)
    sites = inputs.sample_sites(dims, 40, 9)
    assert np.array_equal(oracle.dslash_sites(psi, gauge, dims, sites), full[sites])
    assert np.array_equal(oracle.dslash(psi, gauge, dims, nthreads=1).reshape(-1, 4, 3, 2), full)


def test_l_equals_1_and_2_wrap():
    """x+mu == x-mu (L=2) and x+mu == x (L=1) both follow from the modulo in Eq. 1's deltas."""
    for dims in [(2, 1, 2, 3), (1, 1, 1, 1)]:
        u = random_gauge(dims, 91)
        psi = random_spinor(dims, 92)
        want = (dense_from_eq1(u, dims) @ psi.reshape(-1)).reshape(psi.shape)
        assert np.abs(apply(u, psi, dims) - want).max() < 1e-13

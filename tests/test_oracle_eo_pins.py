"""Pins for the even-odd (checkerboard) oracle functions: oracle.parity_mask, oracle.dslash_parity, oracle.schur_even.

They are restrictions / compositions of the full-lattice operator (itself pinned in test_oracle_pins.py), so the pins here
are what linear algebra fixes about such a decomposition, computed independently with NumPy dense algebra:
  E1  D = D_eo + D_oe, bit for bit (every neighbour of a site has the other parity when all extents are even)
  E2  the dense matrix of schur_even IS the Schur complement  M_ee - M_eo M_oo^{-1} M_oe  of the dense Wilson matrix
  E3  the solution of M x = b obtained with numpy.linalg.solve satisfies the even-odd equations
          Mhat x_e = b_e + D_eo b_o / (2 (4+m)),    x_o = (b_o + D_oe x_e / 2) / (4+m)
      (these are the formulas the CUDA solver dslash_cg_solve_eo implements)
  E4  gamma_5 Mhat gamma_5 = Mhat^dagger, and Mhat^dagger as computed with dagger=True is the conjugate transpose
  E5  det M = (4+m)^{n_odd} det Mhat
"""
import numpy as np
import pytest

import oracle
from paper_2301_03636_b200 import inputs

G5 = np.array([1.0, 1.0, -1.0, -1.0])


def c2r(a):
    return np.ascontiguousarray(np.stack([a.real, a.imag], axis=-1))


def r2c(a):
    return a[..., 0] + 1j * a[..., 1]


def shape4(dims):
    lx, ly, lz, lt = dims
    return (lt, lz, ly, lx)


def rand_spinor(dims, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(shape4(dims) + (4, 3)) + 1j * rng.standard_normal(shape4(dims) + (4, 3))


def dense(fn, dims):
    """matrix of the linear map fn on full-lattice complex spinors, column by column"""
    n = int(np.prod(dims)) * 12
    m = np.empty((n, n), dtype=np.complex128)
    e = np.zeros(n, dtype=np.complex128)
    for k in range(n):
        e[k] = 1.0
        m[:, k] = fn(e.reshape(shape4(dims) + (4, 3))).reshape(-1)
        e[k] = 0.0
    return m


def test_parity_mask_is_the_checkerboard():
    dims = (4, 2, 6, 2)
    odd = oracle.parity_mask(dims)
    assert odd.shape == shape4(dims) and odd.sum() * 2 == odd.size
    for (t, z, y, x), v in np.ndenumerate(odd):
        assert v == bool((x + y + z + t) % 2)


@pytest.mark.parametrize("dims", [(4, 6, 2, 8), (2, 2, 2, 2), (6, 4, 4, 2)])
@pytest.mark.parametrize("dagger", [False, True])
def test_e1_parity_blocks_sum_to_the_full_operator_exactly(dims, dagger):
    u = inputs.gauge_field(dims, 71)
    psi = c2r(rand_spinor(dims, 72))
    full = (oracle.dslash_dagger if dagger else oracle.dslash)(psi, u, dims)
    d_e = oracle.dslash_parity(psi, u, dims, 0, dagger)  # even output from the odd input
    d_o = oracle.dslash_parity(psi, u, dims, 1, dagger)
    odd = oracle.parity_mask(dims)
    assert np.all(d_e[odd] == 0.0) and np.all(d_o[~odd] == 0.0)
    assert np.array_equal(d_e + d_o, full)
    # the input on the output's own parity is ignored
    junk = psi.copy()
    junk[~odd] = 123.0
    assert np.array_equal(oracle.dslash_parity(junk, u, dims, 0, dagger), d_e)


def test_odd_extents_are_refused():
    with pytest.raises(ValueError):
        oracle.dslash_parity(np.zeros((2, 2, 2, 3, 4, 3, 2)), np.zeros((2, 2, 2, 3, 4, 3, 3, 2)), (3, 2, 2, 2), 0)


@pytest.fixture(scope="module")
def small():
    dims = (2, 2, 2, 4)
    mass = 0.15
    u = inputs.gauge_field(dims, 73)
    m_dense = dense(lambda p: r2c(oracle.wilson(c2r(p), u, dims, mass)), dims)
    s_dense = dense(lambda p: r2c(oracle.schur_even(c2r(p), u, dims, mass)), dims)
    sd_dense = dense(lambda p: r2c(oracle.schur_even(c2r(p), u, dims, mass, dagger=True)), dims)
    odd_sites = oracle.parity_mask(dims).reshape(-1)
    odd = np.repeat(odd_sites, 12)  # per complex component, site-major like the flattened spinor
    return dims, mass, u, m_dense, s_dense, sd_dense, odd


def test_e2_schur_even_is_the_schur_complement_of_the_dense_wilson_matrix(small):
    dims, mass, u, m, s, _, odd = small
    ev = ~odd
    mee, meo, moe, moo = m[np.ix_(ev, ev)], m[np.ix_(ev, odd)], m[np.ix_(odd, ev)], m[np.ix_(odd, odd)]
    assert np.abs(moo - (4.0 + mass) * np.eye(moo.shape[0])).max() < 1e-15  # the odd-odd block is (4+m) 1
    schur = mee - meo @ np.linalg.solve(moo, moe)
    assert np.abs(s[np.ix_(ev, ev)] - schur).max() < 1e-13
    # the map ignores odd-site input and returns nothing on odd sites
    assert np.abs(s[np.ix_(odd, odd)]).max() == 0.0 and np.abs(s[np.ix_(ev, odd)]).max() == 0.0 and np.abs(s[np.ix_(odd, ev)]).max() == 0.0


def test_e3_even_odd_equations_reproduce_the_direct_solution(small):
    dims, mass, u, m, s, _, odd = small
    a = 4.0 + mass
    b = rand_spinor(dims, 74)
    x = np.linalg.solve(m, b.reshape(-1)).reshape(b.shape)
    oddm = oracle.parity_mask(dims)[..., None, None]
    b_e, b_o, x_e = b * ~oddm, b * oddm, x * ~oddm
    rhs = b_e + r2c(oracle.dslash_parity(c2r(b_o), u, dims, 0)) / (2.0 * a)
    lhs = r2c(oracle.schur_even(c2r(x_e), u, dims, mass))
    assert np.abs(lhs - rhs).max() < 1e-13
    x_o = (b_o + 0.5 * r2c(oracle.dslash_parity(c2r(x_e), u, dims, 1))) / a
    assert np.abs(x_o - x * oddm).max() < 1e-13


def test_e4_gamma5_hermiticity_and_the_dagger_flag(small):
    dims, mass, u, m, s, sd, odd = small
    assert np.abs(sd - s.conj().T).max() < 1e-13
    g5 = np.tile(np.repeat(G5, 3), int(np.prod(dims)))
    assert np.abs(g5[:, None] * s * g5[None, :] - s.conj().T).max() < 1e-13


def test_e5_determinant_factorisation(small):
    dims, mass, u, m, s, _, odd = small
    ev = ~odd
    sign_m, logdet_m = np.linalg.slogdet(m)
    sign_s, logdet_s = np.linalg.slogdet(s[np.ix_(ev, ev)])
    n_odd = int(odd.sum())
    assert abs(logdet_m - (n_odd * np.log(4.0 + mass) + logdet_s)) < 1e-9
    assert abs(sign_m - sign_s) < 1e-9

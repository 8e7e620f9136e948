"""Host-side checks of the seeded input generator (paper_2301_03636_b200/inputs.py)."""
import numpy as np

from paper_2301_03636_b200 import inputs


def test_links_are_su3_and_row2_is_the_cross_product():
    dims = (4, 6, 2, 3)
    g = inputs.gauge_field(dims, 17)
    u = (g[..., 0] + 1j * g[..., 1]).reshape(-1, 3, 3)
    inputs.check_su3(u)
    assert np.array_equal(u[:, 2, :], np.conj(np.cross(u[:, 0, :], u[:, 1, :])))  # 12-real == 18-real input


def test_haar_moments():
    # For Haar SU(3): E[U_ij] = 0, E|U_ij|^2 = 1/3, E[tr U] = 0, E|tr U|^2 = 1.
    u = inputs.haar_su3(200000, np.random.default_rng(3))
    assert np.abs(u.mean(axis=0)).max() < 5e-3
    assert np.abs((np.abs(u) ** 2).mean(axis=0) - 1.0 / 3.0).max() < 5e-3
    tr = np.trace(u, axis1=1, axis2=2)
    assert abs(tr.mean()) < 1e-2 and abs((np.abs(tr) ** 2).mean() - 1.0) < 2e-2


def test_reproducible_and_chunk_schedule_independent(monkeypatch):
    dims = (8, 8, 8, 4)
    g1, p1 = inputs.fields(dims, 5)
    g2, p2 = inputs.fields(dims, 5)
    assert np.array_equal(g1, g2) and np.array_equal(p1, p2)
    g3, p3 = inputs.fields(dims, 6)
    assert not np.array_equal(p1, p3)
    assert g1.shape == (4, 8, 8, 8, 4, 3, 3, 2) and p1.shape == (4, 8, 8, 8, 4, 3, 2)


def test_spinor_is_standard_normal_per_real():
    p = inputs.spinor_field((8, 8, 8, 8), 9)
    assert abs(p.mean()) < 5e-3 and abs(p.var() - 1.0) < 1e-2


def test_f32_fields_are_rounded_f64_fields():
    dims = (4, 4, 4, 4)
    g64, p64 = inputs.fields(dims, 7, "f64")
    g32, p32 = inputs.fields(dims, 7, "f32")
    assert g32.dtype == np.float32 and np.array_equal(g32, g64.astype(np.float32))
    assert np.array_equal(inputs.promote(p32), p64.astype(np.float32).astype(np.float64))


def test_sample_sites_cover_corners():
    dims = (4, 6, 8, 10)
    s = inputs.sample_sites(dims, 100, 1)
    v = inputs.volume(dims)
    assert s.min() == 0 and s.max() == v - 1 and len(np.unique(s)) == len(s)

"""Seeded synthetic lattice fields (serves tests, bench.py and smoke(); holds none of Dslash's arithmetic).

The paper's workload is a lattice-QCD gauge configuration plus a fermion vector which it never
provides (it names only the sizes 16^4, and 32x32x32x16).  BASELINE.json's
configs replace it by seeded synthetic fields of the same shape and value range, generated here on the
host with NumPy and handed unchanged to both the oracle and the CUDA library:

  * links  U_mu(x): Haar-random SU(3).  Z = (A + iB)/sqrt(2) with A, B ~ N(0,1); the columns of Z are
    orthonormalised by Gram-Schmidt (the QR factor with R_ii > 0, so there is no LAPACK sign
    ambiguity), run twice so the result is unitary to ~1e-16; the matrix is multiplied by
    exp(-i arg(det)/3) so det = 1; finally row 2 is overwritten with conj(row0 x row1), which for an
    SU(3) matrix changes nothing but rounding and makes the 18-real and the 12-real (rows 0,1 only)
    representations of the input the *same* matrix to the last bit of rows 0,1.
  * spinor psi(x)[a][c]: re and im each i.i.d. N(0,1).

Generation is chunked over sites with one independent, seeded stream per (seed, field, chunk), so a
field is reproducible whatever the chunk schedule, and memory stays bounded for 48^3 x 96.

Canonical layout: dims = (L_X, L_Y, L_Z, L_T), x fastest:
    gauge  float64 [L_T, L_Z, L_Y, L_X, 4(mu), 3(row), 3(col), 2(re,im)]
    spinor float64 [L_T, L_Z, L_Y, L_X, 4(spin), 3(colour), 2(re,im)]
"""
from __future__ import annotations

import concurrent.futures
import os

import numpy as np

BASE_SEED = 230103636  # arXiv id of the paper; config k uses BASE_SEED + k
CHUNK_SITES = 1 << 15

_STREAM_GAUGE = 1
_STREAM_SPINOR = 2


def _rng(seed: int, stream: int, chunk: int) -> np.random.Generator:
    return np.random.default_rng([int(seed), int(stream), int(chunk)])


def volume(dims) -> int:
    lx, ly, lz, lt = (int(d) for d in dims)
    return lx * ly * lz * lt


def haar_su3(n: int, rng: np.random.Generator) -> np.ndarray:
    """n Haar-random SU(3) matrices, complex128 [n, 3, 3]."""
    g = rng.standard_normal((n, 3, 3, 2))
    z = (g[..., 0] + 1j * g[..., 1]) / np.sqrt(2.0)
    q = z
    for _ in range(2):  # Gram-Schmidt on the columns, twice
        cols = []
        for k in range(3):
            v = q[:, :, k].copy()
            for u in cols:
                v -= u * np.sum(np.conj(u) * v, axis=1, keepdims=True)
            v /= np.sqrt(np.sum(np.abs(v) ** 2, axis=1, keepdims=True))
            cols.append(v)
        q = np.stack(cols, axis=2)
    det = np.linalg.det(q)
    q = q * np.exp(-1j * np.angle(det) / 3.0)[:, None, None]
    r0, r1 = q[:, 0, :], q[:, 1, :]
    q[:, 2, :] = np.conj(np.cross(r0, r1))
    return q


def check_su3(u: np.ndarray, tol: float = 5e-15) -> None:
    """Assert unitarity and det = 1 (the generator's own post-condition)."""
    u = u.reshape(-1, 3, 3)
    eye = np.eye(3)
    err_u = np.abs(u @ np.conj(np.swapaxes(u, 1, 2)) - eye).max()
    err_d = np.abs(np.linalg.det(u) - 1.0).max()
    if not (err_u <= tol and err_d <= tol):
        raise AssertionError("SU(3) generator post-condition failed: |UU^+-1|=%g |det-1|=%g" % (err_u, err_d))


def _map_chunks(fn, nchunks: int) -> None:
    """Run fn(c) for every chunk; chunks are independent (own RNG stream, own output slice), so a
    thread pool changes nothing but the wall time (NumPy releases the GIL in its kernels)."""
    workers = min(nchunks, len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1))
    if workers <= 1:
        for c in range(nchunks):
            fn(c)
        return
    with concurrent.futures.ThreadPoolExecutor(max_workers=workers) as ex:
        list(ex.map(fn, range(nchunks)))


def gauge_field(dims, seed: int, check: bool = True) -> np.ndarray:
    """Haar-random SU(3) links, float64 [L_T, L_Z, L_Y, L_X, 4, 3, 3, 2]."""
    lx, ly, lz, lt = (int(d) for d in dims)
    v = volume(dims)
    out = np.empty((v, 4, 3, 3, 2), dtype=np.float64)

    def one(c):
        s0 = c * CHUNK_SITES
        n = min(CHUNK_SITES, v - s0)
        u = haar_su3(n * 4, _rng(seed, _STREAM_GAUGE, c))
        if check:
            check_su3(u)
        blk = out[s0:s0 + n].reshape(n * 4, 3, 3, 2)
        blk[..., 0] = u.real
        blk[..., 1] = u.imag

    _map_chunks(one, (v + CHUNK_SITES - 1) // CHUNK_SITES)
    return out.reshape(lt, lz, ly, lx, 4, 3, 3, 2)


def spinor_field(dims, seed: int) -> np.ndarray:
    """N(0,1) + i N(0,1) spinor, float64 [L_T, L_Z, L_Y, L_X, 4, 3, 2]."""
    lx, ly, lz, lt = (int(d) for d in dims)
    v = volume(dims)
    out = np.empty((v, 4, 3, 2), dtype=np.float64)

    def one(c):
        s0 = c * CHUNK_SITES
        n = min(CHUNK_SITES, v - s0)
        out[s0:s0 + n] = _rng(seed, _STREAM_SPINOR, c).standard_normal((n, 4, 3, 2))

    _map_chunks(one, (v + CHUNK_SITES - 1) // CHUNK_SITES)
    return out.reshape(lt, lz, ly, lx, 4, 3, 2)


def fields(dims, seed: int, precision: str = "f64", check: bool = True):
    """(gauge, spinor) in the precision the CUDA library will be given.

    precision "f64": float64 arrays.  "f32": generated in float64, rounded once to float32; the oracle
    is given these float32 values promoted back to float64 (`promote`), so parity measures arithmetic
    error only (DESIGN.md Reading R13).
    """
    g = gauge_field(dims, seed, check=check)
    p = spinor_field(dims, seed)
    if precision == "f64":
        return g, p
    if precision == "f32":
        return g.astype(np.float32), p.astype(np.float32)
    raise ValueError("precision must be 'f64' or 'f32'")


def promote(a: np.ndarray) -> np.ndarray:
    """float64 view/copy of a field for the oracle."""
    return np.ascontiguousarray(a, dtype=np.float64)


def sample_sites(dims, n: int, seed: int) -> np.ndarray:
    """Linear indices of n distinct sampled sites: the 16 lattice corners (every wrap case) plus
    seeded uniform draws.  Used for parity at sizes where the oracle is run site by site."""
    lx, ly, lz, lt = (int(d) for d in dims)
    v = volume(dims)
    corners = []
    for t in (0, lt - 1):
        for z in (0, lz - 1):
            for y in (0, ly - 1):
                for x in (0, lx - 1):
                    corners.append(x + lx * (y + ly * (z + lz * t)))
    rng = np.random.default_rng([int(seed), 3, 0])
    draws = rng.integers(0, v, size=max(0, n - len(corners)), dtype=np.int64)
    return np.unique(np.concatenate([np.asarray(corners, dtype=np.int64), draws]))


# ------------------------------------------------------------------ random numbers the cost model draws (passed in as inputs)
def uniforms(seed: int, n: int) -> np.ndarray:
    """n float64 uniforms in [0, 1): the draws behind the Glorot initialisation (the scaling is the method's, not done here)."""
    return np.random.default_rng([int(seed), 11, 0]).random(int(n))


def permutations(seed: int, epochs: int, n: int) -> np.ndarray:
    """int32 [epochs, n]: the order in which the n training rows are visited in each epoch."""
    rng = np.random.default_rng([int(seed), 12, 0])
    return np.stack([rng.permutation(int(n)) for _ in range(int(epochs))]).astype(np.int32)

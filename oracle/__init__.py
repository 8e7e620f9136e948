"""CPU oracle for the Wilson Dslash operator -- TEST INFRASTRUCTURE ONLY.

ctypes front-end of oracle/dslash_oracle.c (the plain-definition fp64 operator, PAPER.md:47-54,
Eq. 1).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package; the product (paper_2301_03636_b200/) never does, and this package never
imports the product.

Arrays are NumPy, canonical layout:
    spinor  float64 [T, Z, Y, X, 4, 3, 2]      (s = x + L_X*(y + L_Y*(z + L_Z*t)), x fastest)
    gauge   float64 [T, Z, Y, X, 4, 3, 3, 2]   ([mu][row i][col j][re/im])
dims is always (L_X, L_Y, L_Z, L_T).
"""
import ctypes
import os

import numpy as np

from . import build as _build

_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        path = _build.build()
        lib = ctypes.CDLL(path)
        dbl_p = ctypes.POINTER(ctypes.c_double)
        int_p = ctypes.POINTER(ctypes.c_int)
        lib.oracle_gamma.argtypes = [ctypes.c_int, dbl_p]
        lib.oracle_gamma.restype = None
        lib.oracle_dslash.argtypes = [dbl_p, dbl_p, dbl_p, int_p, ctypes.c_int]
        lib.oracle_dslash.restype = ctypes.c_int
        lib.oracle_dslash_dagger.argtypes = [dbl_p, dbl_p, dbl_p, int_p, ctypes.c_int]
        lib.oracle_dslash_dagger.restype = ctypes.c_int
        lib.oracle_dslash_sites.argtypes = [dbl_p, dbl_p, dbl_p, int_p, ctypes.POINTER(ctypes.c_int64),
                                            ctypes.c_int64, ctypes.c_int]
        lib.oracle_dslash_sites.restype = ctypes.c_int
        lib.oracle_max_threads.argtypes = []
        lib.oracle_max_threads.restype = ctypes.c_int
        _LIB = lib
    return _LIB


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _check(psi, gauge, dims):
    lx, ly, lz, lt = (int(d) for d in dims)
    v = lx * ly * lz * lt
    if psi.dtype != np.float64 or gauge.dtype != np.float64:
        raise TypeError("oracle takes float64 arrays")
    if psi.size != v * 24 or gauge.size != v * 72:
        raise ValueError("array sizes do not match dims")
    psi = np.ascontiguousarray(psi)
    gauge = np.ascontiguousarray(gauge)
    cdims = (ctypes.c_int * 4)(lx, ly, lz, lt)
    return psi, gauge, cdims, (lx, ly, lz, lt), v


def gamma(mu: int) -> np.ndarray:
    """gamma_mu as a complex128 [4, 4] array (DeGrand-Rossi, DESIGN.md Reading R4)."""
    out = np.zeros((4, 4, 2), dtype=np.float64)
    _lib().oracle_gamma(int(mu), _dp(out))
    return out[..., 0] + 1j * out[..., 1]


def dslash(psi: np.ndarray, gauge: np.ndarray, dims, nthreads: int = 0) -> np.ndarray:
    """out = D[gauge] psi on the whole lattice (Eq. 1).  nthreads <= 0: all cores."""
    psi, gauge, cdims, (lx, ly, lz, lt), _ = _check(psi, gauge, dims)
    out = np.empty((lt, lz, ly, lx, 4, 3, 2), dtype=np.float64)
    rc = _lib().oracle_dslash(_dp(out), _dp(psi), _dp(gauge), cdims, int(nthreads))
    if rc != 0:
        raise RuntimeError("oracle_dslash failed: %d" % rc)
    return out


def dslash_dagger(psi: np.ndarray, gauge: np.ndarray, dims, nthreads: int = 0) -> np.ndarray:
    """out = D^dagger[gauge] psi: Eq. 1 with gamma_mu -> -gamma_mu (DESIGN.md Reading R19)."""
    psi, gauge, cdims, (lx, ly, lz, lt), _ = _check(psi, gauge, dims)
    out = np.empty((lt, lz, ly, lx, 4, 3, 2), dtype=np.float64)
    rc = _lib().oracle_dslash_dagger(_dp(out), _dp(psi), _dp(gauge), cdims, int(nthreads))
    if rc != 0:
        raise RuntimeError("oracle_dslash_dagger failed: %d" % rc)
    return out


def wilson(psi: np.ndarray, gauge: np.ndarray, dims, mass: float, dagger: bool = False, nthreads: int = 0) -> np.ndarray:
    """M psi = (4 + mass) psi - D psi / 2 (dagger: with D^dagger): the Wilson matrix whose hopping term is Eq. 1."""
    d = (dslash_dagger if dagger else dslash)(psi, gauge, dims, nthreads)
    return (4.0 + float(mass)) * np.ascontiguousarray(psi, dtype=np.float64).reshape(d.shape) - 0.5 * d


def parity_mask(dims) -> np.ndarray:
    """bool [T, Z, Y, X]: True on the odd sites, (x + y + z + t) mod 2 == 1."""
    lx, ly, lz, lt = (int(d) for d in dims)
    t, z, y, x = np.meshgrid(np.arange(lt), np.arange(lz), np.arange(ly), np.arange(lx), indexing="ij")
    return ((x + y + z + t) & 1).astype(bool)


def dslash_parity(psi: np.ndarray, gauge: np.ndarray, dims, out_parity: int, dagger: bool = False, nthreads: int = 0) -> np.ndarray:
    """The checkerboarded hopping term by its definition: restrict Eq. 1 to input on the sites of parity 1 - out_parity and
    output on the sites of parity out_parity (all extents even, so every neighbour of a site has the other parity):
        D_{p,1-p} = P_p D P_{1-p},   P_p = projector on the sites with (x+y+z+t) mod 2 == p.
    Takes and returns full-lattice arrays; entries outside the respective parity are ignored / returned as 0."""
    if any(int(d) % 2 for d in dims):
        raise ValueError("even-odd decomposition needs even extents")
    odd = parity_mask(dims)
    keep_in = odd if out_parity == 0 else ~odd
    src = np.ascontiguousarray(psi, dtype=np.float64).reshape(odd.shape + (4, 3, 2)) * keep_in[..., None, None, None]
    d = (dslash_dagger if dagger else dslash)(src, gauge, dims, nthreads)
    return d * (~keep_in)[..., None, None, None]


def schur_even(psi: np.ndarray, gauge: np.ndarray, dims, mass: float, dagger: bool = False, nthreads: int = 0) -> np.ndarray:
    """The even-odd preconditioned Wilson matrix on the even sites: the Schur complement of M = (4+m) - D/2 with respect
    to its odd-odd block (4+m)*1,
        Mhat = (4+m) - D_eo D_oe / (4 (4+m))        (dagger: with D^dagger in both factors),
    written as the two restricted applications it is.  Full-lattice arrays; odd-site entries of the result are 0."""
    a = 4.0 + float(mass)
    even = ~parity_mask(dims)
    pe = np.ascontiguousarray(psi, dtype=np.float64).reshape(even.shape + (4, 3, 2)) * even[..., None, None, None]
    t_o = dslash_parity(pe, gauge, dims, 1, dagger, nthreads)   # D_oe psi_e
    t_e = dslash_parity(t_o, gauge, dims, 0, dagger, nthreads)  # D_eo D_oe psi_e
    return a * pe - t_e / (4.0 * a)


def dslash_sites(psi: np.ndarray, gauge: np.ndarray, dims, sites, nthreads: int = 0) -> np.ndarray:
    """(D psi)(s) for the linear site indices `sites`; returns float64 [n, 4, 3, 2]."""
    psi, gauge, cdims, _, _ = _check(psi, gauge, dims)
    sites = np.ascontiguousarray(np.asarray(sites, dtype=np.int64))
    out = np.empty((sites.size, 4, 3, 2), dtype=np.float64)
    rc = _lib().oracle_dslash_sites(_dp(out), _dp(psi), _dp(gauge), cdims,
                                    sites.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)), sites.size, int(nthreads))
    if rc != 0:
        raise RuntimeError("oracle_dslash_sites failed: %d" % rc)
    return out


def max_threads() -> int:
    return int(_lib().oracle_max_threads())

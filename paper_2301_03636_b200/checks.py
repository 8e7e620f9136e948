"""The parity metric (DESIGN.md Reading R10); NumPy only, no operator arithmetic."""
import numpy as np


def parity_error(got, ref) -> float:
    """max_k |g_k - r_k| / max(|r_k|, rms(r)) over complex components k.

    north_star asks for a "max relative component error"; a strict |g-r|/|r| is not satisfiable even
    between two fp64 evaluations that differ only in summation order (components of D psi come
    arbitrarily close to 0), so the denominator is floored at the rms magnitude of the reference.
    got/ref: real arrays [..., 2] (re, im), any matching shape.
    """
    g = np.asarray(got, dtype=np.float64)
    r = np.asarray(ref, dtype=np.float64)
    gc = g[..., 0] + 1j * g[..., 1]
    rc = r[..., 0] + 1j * r[..., 1]
    if rc.size == 0:
        return 0.0
    rms = float(np.sqrt(np.mean(np.abs(rc) ** 2)))
    den = np.maximum(np.abs(rc), rms if rms > 0 else 1.0)
    return float(np.max(np.abs(gc - rc) / den))

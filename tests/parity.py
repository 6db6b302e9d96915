"""Norms used by the GPU-vs-oracle parity tests."""
import numpy as np


def force_scale(x, si, sj, k, r0, alive=None):
    """Per-particle sum of |spring contribution| and the global max force norm (denominators of the Q11 norms)."""
    d = x[sj] - x[si]
    r = np.linalg.norm(d, axis=1)
    mag = np.abs(k * (r - r0))
    if alive is not None:
        mag = mag * alive
    sc = np.zeros(x.shape[0])
    np.add.at(sc, si, mag)
    np.add.at(sc, sj, mag)
    return sc


def check_forces(f_gpu, f_ref, scale, tol=1e-12):
    fmax = np.abs(f_ref).max()
    err_glob = np.abs(f_gpu - f_ref).max() / max(fmax, 1e-300)
    per = np.abs(f_gpu - f_ref).max(axis=1)
    bad = per > tol * np.maximum(scale, fmax)
    assert err_glob <= tol, "global force error %.3e" % err_glob
    assert not bad.any(), "per-particle force error on %d particles" % bad.sum()
    return err_glob

"""Norms used by the GPU-vs-oracle parity tests."""
import numpy as np

EPS = np.finfo(np.float64).eps


def force_scale(x, si, sj, k, r0, alive=None):
    """Per-particle sum of |spring contribution| (denominator of the per-particle Q11 norm)."""
    d = x[sj] - x[si]
    r = np.linalg.norm(d, axis=1)
    mag = np.abs(k * (r - r0))
    if alive is not None:
        mag = mag * alive
    sc = np.zeros(x.shape[0])
    np.add.at(sc, si, mag)
    np.add.at(sc, sj, mag)
    return sc


def conditioning_floor(x, si, sj, k, alive=None, ulps=8.0):
    """Absolute error floor of a spring-force evaluation in fp64.

    The force k (r - r0) is a difference of two O(r0) numbers: a rounding error of a few ulp in r (the sqrt, or the
    r^2 * rsqrt(r^2) form) is an ABSOLUTE force error of k * r * eps per spring, however small the extension is.  At
    extensions of 1e-5 r0 (the first steps of a slow pull) that floor, ~1e-15, is above 1e-12 * |f|.  Per particle:
    ulps * eps * sum_s k_s r_s over its live springs."""
    r = np.linalg.norm(x[sj] - x[si], axis=1)
    mag = k * r
    if alive is not None:
        mag = mag * alive
    fl = np.zeros(x.shape[0])
    np.add.at(fl, si, mag)
    np.add.at(fl, sj, mag)
    return ulps * EPS * fl


def check_forces(f_gpu, f_ref, scale, tol=1e-12, floor=None):
    """Q11: global max-norm error <= tol * max|f| and per-particle error <= tol * (sum of |contributions|), each plus
    the conditioning floor when one is given."""
    fmax = np.abs(f_ref).max()
    fl = 0.0 if floor is None else floor
    per = np.abs(f_gpu - f_ref).max(axis=1)
    err_glob = per.max() / max(fmax, 1e-300)
    assert per.max() <= tol * fmax + np.max(fl), "global force error %.3e (relative to max|f|)" % err_glob
    bad = per > tol * np.maximum(scale, fmax) + fl
    assert not bad.any(), "per-particle force error on %d particles" % bad.sum()
    return err_glob

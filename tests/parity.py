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


def check_forces(f_gpu, f_ref, scale, tol=1e-12, floor=None, label=""):
    """Q11 as written: for EVERY particle p, with per_p = max_c |df_p,c|,
        global norm        per_p <= tol * max|f|                    + floor_p
        per-particle norm  per_p <= tol * sum_s |contribution_s,p|  + floor_p      (the sum is `scale`)
    floor_p = 0 unless a conditioning floor (R4: conditioning_floor above) is passed.  The per-particle bound is NOT relaxed
    to the global one for particles whose own contributions are small: those are the particles it exists for.
    Returns (and prints, for DESIGN.md's table: run pytest with -s) the measured errors: err_glob = max per_p / max|f|,
    err_pp = max per_p / scale_p, err_pp_net = max (per_p - floor_p)+ / scale_p."""
    fmax = np.abs(f_ref).max()
    fl = np.zeros(f_ref.shape[0]) if floor is None else np.broadcast_to(floor, (f_ref.shape[0],))
    per = np.abs(f_gpu - f_ref).max(axis=1)
    err_glob = per.max() / max(fmax, 1e-300)
    live = scale > 0
    err_pp = float((per[live] / scale[live]).max()) if live.any() else 0.0
    err_pp_net = float((np.maximum(per[live] - fl[live], 0.0) / scale[live]).max()) if live.any() else 0.0
    print("check_forces %s: err_glob %.3e  err_pp %.3e  err_pp_net_of_floor %.3e  (N = %d, floor %s)"
          % (label, err_glob, err_pp, err_pp_net, per.size, "R4" if floor is not None else "none"))
    bad_g = per > tol * fmax + fl
    assert not bad_g.any(), "global force error %.3e (relative to max|f|) on %d particles" % (err_glob, bad_g.sum())
    bad = per > tol * scale + fl
    assert not bad.any(), "per-particle force error on %d particles (max %.3e of the particle's own contributions, %.3e net of the floor)" % (
        bad.sum(), err_pp, err_pp_net)
    return err_glob, err_pp, err_pp_net

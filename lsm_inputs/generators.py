"""Synthetic particle-spring networks shaped like the paper's image-derived specimens.

The paper measured on its own "Poisson composite" input files (Table 2), which are not
available; the five configs of BASELINE.json stand in for them.  They keep the paper's structure: 2-D triangular
packing with one particle per pixel, a handful of spring types (Table 1),
grip rows at the top and bottom, optional notch.

Geometry: site (c, r), c in [0,nx), r in [0,ny):
    x = (c + 0.5*(r mod 2))*r0,  y = r*(sqrt(3)/2)*r0,  id = r*nx + c   (before removed sites are compacted away)
Springs per site, in this caller order: E (c,r)-(c+1,r); N (c,r)-(c,r+1); D: even r (c,r)-(c-1,r+1), odd r (c,r)-(c+1,r+1).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

FIXED, MOVE = 0, 1
SQ3_2 = np.sqrt(3.0) / 2.0


@dataclass
class BoundaryGroup:
    ids: np.ndarray          # int32 particle ids (caller numbering)
    mode: int                # FIXED or MOVE
    du: np.ndarray           # displacement per step, [2]


@dataclass
class Problem:
    name: str
    x: np.ndarray            # [N,2] float64
    v: np.ndarray            # [N,2] float64
    spring_i: np.ndarray     # [M] int32
    spring_j: np.ndarray     # [M] int32
    k: np.ndarray            # [M] float64
    r0: np.ndarray           # [M] float64
    rc: np.ndarray           # [M] float64  (absolute length)
    dt: float
    gamma: float
    groups: List[BoundaryGroup] = field(default_factory=list)
    mass: float = 1.0
    n_batch: int = 1
    particle_offsets: Optional[np.ndarray] = None   # [n_batch+1] int64
    spring_offsets: Optional[np.ndarray] = None     # [n_batch+1] int64
    sample_every: int = 100
    steps: int = 0           # the run length BASELINE.json names
    meta: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.x.shape[0])

    @property
    def M(self) -> int:
        return int(self.spring_i.shape[0])


def triangular_lattice(nx: int, ny: int, r0: float = 1.0, keep: Optional[np.ndarray] = None):
    """Particles and nearest-neighbour springs of an nx-by-ny triangular packing.

    keep: optional bool [ny,nx]; sites with keep=False (and every spring touching them) are removed and the
    remaining particles are numbered in row-major order.  Returns (x[N,2], spring_i, spring_j, site_of_particle[N],
    spring_kind[M] in {0:E,1:N,2:D}).  A full lattice has ny(nx-1) + (ny-1)(2nx-1) springs.
    """
    if keep is None:
        keep = np.ones((ny, nx), dtype=bool)
    keep = np.asarray(keep, dtype=bool)
    assert keep.shape == (ny, nx)
    pid = np.full(ny * nx, -1, dtype=np.int64)
    flat = keep.ravel()
    n = int(flat.sum())
    pid[flat] = np.arange(n, dtype=np.int64)
    pid = pid.reshape(ny, nx)

    c = np.arange(nx, dtype=np.float64)[None, :]
    r = np.arange(ny, dtype=np.int64)[:, None]
    xs = (c + 0.5 * (r % 2)) * r0 + np.zeros((ny, 1))
    ys = (r * SQ3_2 * r0) + np.zeros((1, nx))
    x = np.stack([xs[keep], ys[keep]], axis=1)

    # neighbour site tables, slot order E, N, D per site
    a = np.full((ny, nx, 3), -1, dtype=np.int64)     # partner particle id, -1 if none
    a[:, :-1, 0] = pid[:, 1:]                        # E
    a[:-1, :, 1] = pid[1:, :]                        # N
    ev = np.arange(0, ny - 1, 2)                     # even rows: (c-1, r+1)
    od = np.arange(1, ny - 1, 2)                     # odd rows:  (c+1, r+1)
    a[ev[:, None], np.arange(1, nx)[None, :], 2] = pid[ev[:, None] + 1, np.arange(0, nx - 1)[None, :]]
    a[od[:, None], np.arange(0, nx - 1)[None, :], 2] = pid[od[:, None] + 1, np.arange(1, nx)[None, :]]
    own = np.broadcast_to(pid[:, :, None], a.shape)
    ok = (a >= 0) & (own >= 0)
    si = own[ok].astype(np.int32)
    sj = a[ok].astype(np.int32)
    kind = np.broadcast_to(np.arange(3, dtype=np.int8)[None, None, :], a.shape)[ok]
    site = np.flatnonzero(flat).astype(np.int64)
    return x, si, sj, site, kind


def blob_image(nx: int, ny: int, n_blobs: int, sigma_lo: float, sigma_hi: float, frac_stiff: float, seed: int):
    """Seeded sum of Gaussian blobs, thresholded so that `frac_stiff` of the pixels are stiff (True)."""
    rng = np.random.default_rng(seed)
    cx = rng.uniform(0, nx, n_blobs)
    cy = rng.uniform(0, ny, n_blobs)
    sg = rng.uniform(sigma_lo, sigma_hi, n_blobs)
    px = np.arange(nx, dtype=np.float64)[None, :]
    py = np.arange(ny, dtype=np.float64)[:, None]
    fld = np.zeros((ny, nx))
    for b in range(n_blobs):
        fld += np.exp(-((px - cx[b]) ** 2 + (py - cy[b]) ** 2) / (2.0 * sg[b] ** 2))
    thr = np.quantile(fld, 1.0 - frac_stiff)
    return fld > thr


def _hmean(a, b):
    return np.where(a == b, a, 2.0 * a * b / (a + b))


def two_phase_spring_params(stiff_of_particle, si, sj, k_stiff, k_soft, rcr_stiff, rcr_soft, r0=1.0):
    """Per-spring k and rc from per-particle phase; interface springs take the harmonic mean (BASELINE.json cfg 2)."""
    kp = np.where(stiff_of_particle, k_stiff, k_soft).astype(np.float64)
    rp = np.where(stiff_of_particle, rcr_stiff, rcr_soft).astype(np.float64)
    k = _hmean(kp[si], kp[sj])
    rc = _hmean(rp[si], rp[sj]) * r0
    return k, rc


def porous_keep_mask(nx, ny, porosity, rad_lo, rad_hi, seed, guard_rows=3, r0=1.0):
    """Seeded random circular voids removed until >= porosity of all sites are gone; guard rows stay solid."""
    rng = np.random.default_rng(seed)
    keep = np.ones((ny, nx), dtype=bool)
    W, H = nx * r0, (ny - 1) * SQ3_2 * r0
    target = int(np.ceil(porosity * nx * ny))
    removed = 0
    n_voids = 0
    rows_y = np.arange(ny) * SQ3_2 * r0
    while removed < target:
        cx, cy, rad = rng.uniform(0, W), rng.uniform(0, H), rng.uniform(rad_lo, rad_hi) * r0
        r_lo = max(guard_rows, int(np.floor((cy - rad) / (SQ3_2 * r0))))
        r_hi = min(ny - guard_rows - 1, int(np.ceil((cy + rad) / (SQ3_2 * r0))))
        c_lo = max(0, int(np.floor(cx - rad - 1)))
        c_hi = min(nx - 1, int(np.ceil(cx + rad + 1)))
        n_voids += 1
        if r_hi < r_lo or c_hi < c_lo:
            continue
        rr = np.arange(r_lo, r_hi + 1)
        cc = np.arange(c_lo, c_hi + 1)
        sx = (cc[None, :] + 0.5 * (rr[:, None] % 2)) * r0
        sy = rows_y[rr][:, None]
        inside = (sx - cx) ** 2 + (sy - cy) ** 2 <= rad * rad
        sub = keep[r_lo:r_hi + 1, c_lo:c_hi + 1]
        removed += int((sub & inside).sum())
        sub &= ~inside
    return keep, n_voids


def velocity_ramp(x, du_y, dt, y_top):
    """Linear initial velocity ramp v_y = (y/y_top) * du_y/dt (avoids a grip shock at step 0)."""
    v = np.zeros_like(x)
    v[:, 1] = (x[:, 1] / y_top) * (du_y / dt)
    return v


def _grips(x, site, nx, ny, du_y):
    row = site // nx
    bot = np.flatnonzero(row == 0).astype(np.int32)
    top = np.flatnonzero(row == ny - 1).astype(np.int32)
    return [BoundaryGroup(bot, FIXED, np.zeros(2)), BoundaryGroup(top, MOVE, np.array([0.0, du_y]))]


def _meta(nx, ny, r0, n_top):
    return dict(nx=nx, ny=ny, r0=r0, W0=n_top * r0, H0=(ny - 1) * SQ3_2 * r0)


def config1(nx: int = 64, ny: int = 64) -> Problem:
    """BASELINE.json configs[0]: 64x64 lattice, k=1, rc=1.1, dt=0.01, top pulled 1e-4/step, gamma=0.01, 10^4 steps."""
    x, si, sj, site, _ = triangular_lattice(nx, ny)
    M = si.size
    g = _grips(x, site, nx, ny, 1e-4)
    return Problem("cfg1_lattice%dx%d" % (nx, ny), x, np.zeros_like(x), si, sj, np.full(M, 1.0), np.full(M, 1.0),
                   np.full(M, 1.1), 0.01, 0.01, g, steps=10000, meta=_meta(nx, ny, 1.0, g[1].ids.size))


def config2(n: int = 512, seed: int = 20220104, n_blobs: int = 200, du_y: Optional[float] = None) -> Problem:
    """BASELINE.json configs[1]: two-phase composite from a seeded blob image (40 % stiff), k 10/1, rc 1.05/1.2."""
    s = n / 512.0
    stiff = blob_image(n, n, n_blobs, 8.0 * s, 32.0 * s, 0.40, seed)
    x, si, sj, site, _ = triangular_lattice(n, n)
    k, rc = two_phase_spring_params(stiff.ravel()[site], si, sj, 10.0, 1.0, 1.05, 1.2)
    dt = 0.05
    H0 = (n - 1) * SQ3_2
    if du_y is None:
        du_y = 1.5e-6 * H0
    g = _grips(x, site, n, n, du_y)
    v = velocity_ramp(x, du_y, dt, H0)
    v[g[0].ids] = 0.0
    m = _meta(n, n, 1.0, g[1].ids.size)
    m["stiff_fraction"] = float(stiff.mean())
    return Problem("cfg2_twophase%d" % n, x, v, si, sj, k, np.ones_like(k), rc, dt, 0.01, g, steps=50000, meta=m)


def config3(n: int = 2048, seed: int = 12345, porosity: float = 0.30, strain_per_step: float = 1e-6) -> Problem:
    """BASELINE.json configs[2]: porous lattice, seeded circular voids (radius U[5,40] sites, scaled with n/2048),
    k=1, rc per spring ~ U[1.05,1.15].  The bench workload (HBM-bound)."""
    s = max(n / 2048.0, 0.125)
    keep, n_voids = porous_keep_mask(n, n, porosity, 5.0 * s if n < 2048 else 5.0, 40.0 * s if n < 2048 else 40.0, seed)
    x, si, sj, site, _ = triangular_lattice(n, n, keep=keep)
    M = si.size
    rc = np.random.default_rng(seed + 1).uniform(1.05, 1.15, M)
    dt = 0.05
    H0 = (n - 1) * SQ3_2
    du_y = strain_per_step * H0
    g = _grips(x, site, n, n, du_y)
    v = velocity_ramp(x, du_y, dt, H0)
    v[g[0].ids] = 0.0
    m = _meta(n, n, 1.0, g[1].ids.size)
    m.update(n_voids=n_voids, porosity=1.0 - x.shape[0] / float(n * n))
    return Problem("cfg3_porous%d" % n, x, v, si, sj, np.ones(M), np.ones(M), rc, dt, 0.01, g, steps=2000, meta=m)


def single_specimen(b: int, n: int = 128, du_y: float = 3.3e-4, dt: float = 0.03) -> Problem:
    """Specimen b of BASELINE.json configs[3] on its own (image seed 1000+b, stiffness ratio from {2,5,10,20})."""
    rng = np.random.default_rng(1000 + b)
    ratio = float(np.array([2.0, 5.0, 10.0, 20.0])[rng.integers(4)])
    frac = float(rng.uniform(0.4, 0.6))
    stiff = blob_image(n, n, 50, 2.0, 8.0, frac, 1_000_000 + b)
    x, si, sj, site, _ = triangular_lattice(n, n)
    k, rc = two_phase_spring_params(stiff.ravel()[site], si, sj, ratio, 1.0, 1.05, 1.2)
    H0 = (n - 1) * SQ3_2
    g = _grips(x, site, n, n, du_y)
    v = velocity_ramp(x, du_y, dt, H0)
    v[g[0].ids] = 0.0
    m = _meta(n, n, 1.0, g[1].ids.size)
    m["ratio"] = ratio
    return Problem("cfg4_specimen%d" % b, x, v, si, sj, k, np.ones_like(k), rc, dt, 0.01, g, steps=20000, meta=m)


def config4(B: int = 1024, n: int = 128, first: int = 0) -> Problem:
    """BASELINE.json configs[3]: B independent n-by-n two-phase specimens as one disjoint union (batched layout)."""
    parts = [single_specimen(first + b, n) for b in range(B)]
    po = np.zeros(B + 1, dtype=np.int64)
    so = np.zeros(B + 1, dtype=np.int64)
    for b, p in enumerate(parts):
        po[b + 1] = po[b] + p.N
        so[b + 1] = so[b] + p.M
    x = np.concatenate([p.x for p in parts])
    v = np.concatenate([p.v for p in parts])
    si = np.concatenate([p.spring_i + np.int32(po[b]) for b, p in enumerate(parts)]).astype(np.int32)
    sj = np.concatenate([p.spring_j + np.int32(po[b]) for b, p in enumerate(parts)]).astype(np.int32)
    k = np.concatenate([p.k for p in parts])
    rc = np.concatenate([p.rc for p in parts])
    groups = []
    for gi in range(2):
        ids = np.concatenate([p.groups[gi].ids + np.int32(po[b]) for b, p in enumerate(parts)]).astype(np.int32)
        groups.append(BoundaryGroup(ids, parts[0].groups[gi].mode, parts[0].groups[gi].du))
    m = dict(parts[0].meta)
    m["ratios"] = [p.meta["ratio"] for p in parts]
    return Problem("cfg4_batch%dx%d" % (B, n), x, v, si, sj, k, np.ones_like(k), rc, parts[0].dt, 0.01, groups,
                   n_batch=B, particle_offsets=po, spring_offsets=so, steps=20000, meta=m)


def config5(n: int = 8192, eps0: float = 0.025, notch_frac: float = 0.10) -> Problem:
    """BASELINE.json configs[4]: large uniform lattice with a single edge notch, affine pre-strain eps0, grips held."""
    x, si, sj, site, kind = triangular_lattice(n, n)
    row_i = site[si] // n
    mid = n // 2 - 1                                   # springs from row mid to row mid+1 cross the notch line
    xm = 0.5 * (x[si, 0] + x[sj, 0])
    cut = (kind != 0) & (row_i == mid) & (xm < notch_frac * n)
    keep = ~cut
    si, sj = si[keep], sj[keep]
    M = si.size
    x = x * np.array([1.0 - eps0 / 3.0, 1.0 + eps0])[None, :]
    g = _grips(x, site, n, n, 0.0)
    g[1].mode = FIXED
    m = _meta(n, n, 1.0, g[1].ids.size)
    m.update(eps0=eps0, n_cut=int(cut.sum()))
    return Problem("cfg5_notch%d" % n, x, np.zeros_like(x), si, sj, np.ones(M), np.ones(M), np.full(M, 1.1), 0.05, 0.01,
                   g, steps=5000, meta=m)


def shuffle_ids(p: Problem, seed: int) -> Problem:
    """Randomly renumber particles, permute spring order and swap endpoints: imitates an arbitrary input-file order."""
    assert p.n_batch == 1
    rng = np.random.default_rng(seed)
    perm = rng.permutation(p.N)                        # new id -> old id
    inv = np.empty_like(perm)
    inv[perm] = np.arange(p.N)
    sp = rng.permutation(p.M)
    si, sj = inv[p.spring_i[sp]].astype(np.int32), inv[p.spring_j[sp]].astype(np.int32)
    sw = rng.random(p.M) < 0.5
    si, sj = np.where(sw, sj, si).astype(np.int32), np.where(sw, si, sj).astype(np.int32)
    groups = [BoundaryGroup(inv[g.ids].astype(np.int32), g.mode, g.du.copy()) for g in p.groups]
    q = Problem(p.name + "_shuffled", p.x[perm].copy(), p.v[perm].copy(), si, sj, p.k[sp].copy(), p.r0[sp].copy(),
                p.rc[sp].copy(), p.dt, p.gamma, groups, mass=p.mass, sample_every=p.sample_every, steps=p.steps,
                meta=dict(p.meta))
    q.meta["perm"] = perm          # new particle id -> old particle id
    q.meta["spring_perm"] = sp     # new spring id -> old spring id
    return q


def cubic_lattice_3d(nx: int, ny: int, nz: int, r0: float = 1.0, diagonals: bool = True):
    """3-D test network (the paper's kernel listing is 3-D): simple cubic sites with springs to the
    +x, +y, +z neighbours (rest length r0) and, optionally, the face diagonals in the xy, yz and zx planes (rest length
    sqrt(2) r0) that make the network rigid.  Returns x [N,3], spring_i, spring_j, r0_s."""
    ix, iy, iz = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    idx = (ix * ny + iy) * nz + iz
    x = np.stack([ix, iy, iz], axis=-1).reshape(-1, 3).astype(np.float64) * r0
    si, sj, rr = [], [], []

    def link(a, b, length):
        si.append(a.ravel()); sj.append(b.ravel()); rr.append(np.full(a.size, length))

    link(idx[:-1], idx[1:], r0); link(idx[:, :-1], idx[:, 1:], r0); link(idx[:, :, :-1], idx[:, :, 1:], r0)
    if diagonals:
        s2 = np.sqrt(2.0) * r0
        link(idx[:-1, :-1], idx[1:, 1:], s2); link(idx[:-1, 1:], idx[1:, :-1], s2)
        link(idx[:, :-1, :-1], idx[:, 1:, 1:], s2); link(idx[:, :-1, 1:], idx[:, 1:, :-1], s2)
        link(idx[:-1, :, :-1], idx[1:, :, 1:], s2); link(idx[1:, :, :-1], idx[:-1, :, 1:], s2)
    return x, np.concatenate(si).astype(np.int32), np.concatenate(sj).astype(np.int32), np.concatenate(rr)


def config3d(n: int = 128, strain_per_step: float = 1e-6) -> Problem:
    """A 3-D workload for the D = 3 path (not a BASELINE.json config: those are all 2-D): n^3 cubic network with face
    diagonals, k = 1, rc = 1.1 x rest length, bottom face (z = 0) fixed, top face pulled in +z, velocity ramp."""
    x, si, sj, r0 = cubic_lattice_3d(n, n, n)
    M = si.size
    dt = 0.02
    H0 = float(n - 1)
    du = np.array([0.0, 0.0, strain_per_step * H0])
    iz = np.round(x[:, 2]).astype(int)
    bot = np.flatnonzero(iz == 0).astype(np.int32)
    top = np.flatnonzero(iz == n - 1).astype(np.int32)
    v = np.zeros_like(x)
    v[:, 2] = (x[:, 2] / H0) * (du[2] / dt)
    v[bot] = 0.0
    g = [BoundaryGroup(bot, FIXED, np.zeros(3)), BoundaryGroup(top, MOVE, du)]
    return Problem("cube3d_%d" % n, x, v, si, sj, np.ones(M), r0, 1.1 * r0, dt, 0.01, g, steps=2000,
                   meta=dict(nx=n, ny=n, nz=n, r0=1.0, W0=float(n * n), H0=H0))

"""ctypes driver for the CPU oracle (oracle/olsm.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
It builds liboracle_lsm.so with gcc (-O2 -ffp-contract=off: no FMA contraction, IEEE sqrt and divide) on first use.
Nothing here is shared with, or imported by, paper_2201_04565_b200/.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle_lsm.so")
_SRC = os.path.join(_HERE, "olsm.c")
_lib = None
MAX_GROUPS = 8


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


def _p(a, t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        d, i32, i64, u8 = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_uint8)
        L.olsm_create.restype = C.c_void_p
        L.olsm_create.argtypes = [C.c_int32, C.c_int64, C.c_int64, C.c_int32, i64, i64, d, d, d, C.c_double,
                                  i32, i32, d, d, d, C.c_double, C.c_double, C.c_int32]
        L.olsm_set_boundary.argtypes = [C.c_void_p, C.c_int32, i32, C.c_int64, C.c_int32, d]
        L.olsm_step.argtypes = [C.c_void_p, C.c_int64]
        L.olsm_set_threads.argtypes = [C.c_void_p, C.c_int32]
        L.olsm_write_state.argtypes = [C.c_void_p, d, d]
        L.olsm_read_state.argtypes = [C.c_void_p, d, d]
        L.olsm_read_forces.argtypes = [C.c_void_p, d]
        L.olsm_read_broken.argtypes = [C.c_void_p, u8, i64, i64]
        L.olsm_read_energy.argtypes = [C.c_void_p, d, d]
        L.olsm_read_virial.argtypes = [C.c_void_p, d]
        L.olsm_read_strain.argtypes = [C.c_void_p, d, u8]
        L.olsm_read_stress.argtypes = [C.c_void_p, C.c_int64, i64, i64, d, d, d, i64]
        L.olsm_n_samples.restype = C.c_int64
        L.olsm_n_samples.argtypes = [C.c_void_p]
        L.olsm_current_step.restype = C.c_int64
        L.olsm_current_step.argtypes = [C.c_void_p]
        L.olsm_destroy.argtypes = [C.c_void_p]
        L.olsm_destroy.restype = None
        _lib = L
    return _lib


class OracleSim:
    """Thin handle around olsm_*.  Arrays in and out use the caller's numbering, x/v/f as [N,D] float64."""

    def __init__(self, x, spring_i, spring_j, k, r0, rc, dt, gamma=0.0, v=None, mass=1.0, n_batch=1,
                 particle_offsets=None, spring_offsets=None, sample_every=0):
        L = lib()
        x = np.ascontiguousarray(x, dtype=np.float64)
        self.N, self.D = x.shape
        self.M = int(len(spring_i))
        self.B = int(n_batch)
        v = None if v is None else np.ascontiguousarray(v, dtype=np.float64)
        marr = None
        mu = 1.0
        if np.ndim(mass) == 0:
            mu = float(mass)
        else:
            marr = np.ascontiguousarray(mass, dtype=np.float64)
        si = np.ascontiguousarray(spring_i, dtype=np.int32)
        sj = np.ascontiguousarray(spring_j, dtype=np.int32)
        bc = lambda a: np.ascontiguousarray(np.broadcast_to(np.asarray(a, dtype=np.float64), (self.M,)))
        po = None if particle_offsets is None else np.ascontiguousarray(particle_offsets, dtype=np.int64)
        so = None if spring_offsets is None else np.ascontiguousarray(spring_offsets, dtype=np.int64)
        self._h = L.olsm_create(self.D, self.N, self.M, self.B, _p(po, C.c_int64), _p(so, C.c_int64),
                                _p(x, C.c_double), _p(v, C.c_double), _p(marr, C.c_double), mu,
                                _p(si, C.c_int32), _p(sj, C.c_int32), _p(bc(k), C.c_double), _p(bc(r0), C.c_double),
                                _p(bc(rc), C.c_double), float(dt), float(gamma), int(sample_every))
        if not self._h:
            raise ValueError("olsm_create rejected the inputs")

    @classmethod
    def from_problem(cls, p, sample_every=None, gamma=None):
        s = cls(p.x, p.spring_i, p.spring_j, p.k, p.r0, p.rc, p.dt, p.gamma if gamma is None else gamma, v=p.v,
                mass=p.mass, n_batch=p.n_batch, particle_offsets=p.particle_offsets, spring_offsets=p.spring_offsets,
                sample_every=p.sample_every if sample_every is None else sample_every)
        for gi, g in enumerate(p.groups):
            s.set_boundary(gi, g.ids, g.mode, g.du)
        return s

    def set_boundary(self, group, ids, mode, du=None):
        ids = np.ascontiguousarray(ids, dtype=np.int32)
        du = np.zeros(self.D) if du is None else np.ascontiguousarray(du, dtype=np.float64)
        rc = lib().olsm_set_boundary(self._h, int(group), _p(ids, C.c_int32), ids.size, int(mode), _p(du, C.c_double))
        if rc != 0:
            raise ValueError("olsm_set_boundary failed: %d" % rc)

    def step(self, n=1):
        if lib().olsm_step(self._h, int(n)) != 0:
            raise ValueError("olsm_step failed")

    def set_threads(self, n):
        """n > 1: the all-cores timing variant (bit-equal to the serial loop); n <= 1: the serial reference loop."""
        if lib().olsm_set_threads(self._h, int(n)) != 0:
            raise ValueError("olsm_set_threads failed")

    def write_state(self, x, v=None):
        x = np.ascontiguousarray(x, dtype=np.float64)
        v = None if v is None else np.ascontiguousarray(v, dtype=np.float64)
        lib().olsm_write_state(self._h, _p(x, C.c_double), _p(v, C.c_double))

    def read_state(self):
        x = np.empty((self.N, self.D)); v = np.empty((self.N, self.D))
        lib().olsm_read_state(self._h, _p(x, C.c_double), _p(v, C.c_double))
        return x, v

    def read_forces(self):
        f = np.empty((self.N, self.D))
        lib().olsm_read_forces(self._h, _p(f, C.c_double))
        return f

    def read_broken(self):
        b = np.empty(self.M, dtype=np.uint8); bs = np.empty(self.M, dtype=np.int64); n = C.c_int64(0)
        lib().olsm_read_broken(self._h, _p(b, C.c_uint8), _p(bs, C.c_int64), C.byref(n))
        return b.astype(bool), bs, int(n.value)

    def read_energy(self):
        U = np.empty(self.B); KE = np.empty(self.B)
        lib().olsm_read_energy(self._h, _p(U, C.c_double), _p(KE, C.c_double))
        return U, KE

    def read_virial(self):
        """Per-particle virial (Eq. 7 without 1/Omega): [N,3] = S_xx, S_yy, S_xy; 3-D: [N,6] = xx, yy, zz, xy, yz, zx."""
        S = np.empty((self.N, 3 if self.D == 2 else 6))
        if lib().olsm_read_virial(self._h, _p(S, C.c_double)) != 0:
            raise ValueError("olsm_read_virial failed")
        return S

    def read_strain(self):
        """Per-particle Lagrangian strain (Eq. 8, reading Q21): ([N,3] = e_xx, e_yy, e_xy; 3-D: [N,6] = xx, yy, zz, xy, yz,
        zx), ok[N] bool (False: fewer than D independent bonds, strain reported as 0)."""
        E = np.empty((self.N, 3 if self.D == 2 else 6)); ok = np.empty(self.N, dtype=np.uint8)
        if lib().olsm_read_strain(self._h, _p(E, C.c_double), _p(ok, C.c_uint8)) != 0:
            raise ValueError("olsm_read_strain failed")
        return E, ok.astype(bool)

    @property
    def current_step(self):
        return int(lib().olsm_current_step(self._h))

    def read_stress(self):
        """Returns dict(step[ns], R[ns,B,8,D], U[ns,B], KE[ns,B], n_broken[ns,B]) and clears the history."""
        ns = int(lib().olsm_n_samples(self._h))
        step = np.empty(ns, dtype=np.int64); R = np.empty((ns, self.B, MAX_GROUPS, self.D))
        U = np.empty((ns, self.B)); KE = np.empty((ns, self.B)); nb = np.empty((ns, self.B), dtype=np.int64)
        n = C.c_int64(0)
        lib().olsm_read_stress(self._h, ns, C.byref(n), _p(step, C.c_int64), _p(R, C.c_double), _p(U, C.c_double),
                               _p(KE, C.c_double), _p(nb, C.c_int64))
        return dict(step=step, R=R, U=U, KE=KE, n_broken=nb)

    def close(self):
        if getattr(self, "_h", None):
            lib().olsm_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

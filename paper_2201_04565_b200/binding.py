"""ctypes binding of include/lsm.h -- same names as the C ABI, argument marshalling only.

Every step of the path runs inside liblsm_b200.so.  PyTorch is used for plumbing only: its caching allocator backs
the library's device memory (through the lsm_desc.alloc / free_ callbacks) and its current CUDA stream is the stream
the kernels are enqueued on.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

FIXED, MOVE = 0, 1
FORCE_AUTO, FORCE_SCATTER, FORCE_GATHER, FORCE_SCATTER_WARP, FORCE_SCATTER_TILE = 0, 1, 2, 3, 4
REORDER_NONE, REORDER_MORTON, REORDER_RCM, REORDER_BLOCKED = 0, 1, 2, 3
GATHER_AUTO, GATHER_DIRECT, GATHER_STREAMED = 0, 1, 2
WINDOW_AUTO, WINDOW_ON, WINDOW_OFF = 0, 1, 2
FUSION_AUTO, FUSION_ON, FUSION_OFF, FUSION_RESIDENT = 0, 1, 2, 3
MAX_GROUPS = 8

EXPORTS = ["lsm_create", "lsm_set_boundary", "lsm_step", "lsm_write_state", "lsm_read_state", "lsm_read_forces",
           "lsm_read_broken", "lsm_read_energy", "lsm_read_virial", "lsm_read_strain", "lsm_read_stress", "lsm_run_to_failure", "lsm_set_strain_rate", "lsm_compact", "lsm_sync", "lsm_get_info",
           "lsm_device_state", "lsm_last_error", "lsm_destroy", "lsm_abi_version", "lsm_spring_energy_static"]
STATIC_MAX_SPRINGS = 1 << 28

_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class LsmDesc(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("dim", C.c_int32), ("n_particles", C.c_int64), ("n_springs", C.c_int64),
        ("n_batch", C.c_int32), ("_pad0", C.c_int32),
        ("particle_offsets", C.POINTER(C.c_int64)), ("spring_offsets", C.POINTER(C.c_int64)),
        ("x", C.POINTER(C.c_double)), ("v", C.POINTER(C.c_double)), ("mass", C.POINTER(C.c_double)),
        ("mass_uniform", C.c_double),
        ("spring_i", C.POINTER(C.c_int32)), ("spring_j", C.POINTER(C.c_int32)),
        ("k", C.POINTER(C.c_double)), ("r0", C.POINTER(C.c_double)), ("rc", C.POINTER(C.c_double)),
        ("k_uniform", C.c_double), ("r0_uniform", C.c_double), ("rc_uniform", C.c_double),
        ("dt", C.c_double), ("gamma", C.c_double),
        ("sample_every", C.c_int32), ("history_capacity", C.c_int32), ("compact_every", C.c_int32),
        ("reorder", C.c_int32), ("force_mode", C.c_int32), ("exact", C.c_int32), ("step_fusion", C.c_int32),
        ("gather_variant", C.c_int32), ("gather_window", C.c_int32), ("device", C.c_int32), ("_pad1", C.c_int32), ("cluster_size", C.c_int32),
        ("stream", C.c_void_p),
        ("alloc", _ALLOC_FN), ("free_", _FREE_FN), ("alloc_user", C.c_void_p),
    ]


class LsmInfo(C.Structure):
    _fields_ = [
        ("n_particles", C.c_int64), ("n_springs", C.c_int64), ("n_half_edges_stored", C.c_int64),
        ("bytes_per_half_edge", C.c_int64), ("param_mode", C.c_int32), ("n_types", C.c_int32),
        ("force_mode", C.c_int32), ("exact", C.c_int32), ("reorder", C.c_int32), ("n_batch", C.c_int32),
        ("device_bytes", C.c_int64), ("kernels_launched", C.c_int64), ("current_step", C.c_int64),
        ("gather_variant", C.c_int32), ("pipeline_stages", C.c_int32), ("stage_bytes", C.c_int64),
        ("step_fusion", C.c_int32), ("cluster_size", C.c_int32), ("resident_smem_bytes", C.c_int64),
        ("window_particles", C.c_int32), ("window_stages", C.c_int32),
    ]


class LsmError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("lsm status %d: %s" % (status, msg))
        self.status = status


_lib = None


def library_path() -> str:
    return _build.SO


def library():
    """Load liblsm_b200.so (building it in-tree with nvcc if it is missing or stale). Fails loudly if it cannot."""
    global _lib
    if _lib is None:
        so = _build.build()
        if not os.path.exists(so):
            raise LsmError(-4, "liblsm_b200.so is missing and could not be built; there is no fallback path")
        L = C.CDLL(so)
        d, i32, i64, u8 = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_uint8)
        L.lsm_create.argtypes = [C.POINTER(LsmDesc), C.POINTER(C.c_void_p)]
        L.lsm_set_boundary.argtypes = [C.c_void_p, C.c_int32, i32, C.c_int64, C.c_int32, d]
        L.lsm_step.argtypes = [C.c_void_p, C.c_int64]
        L.lsm_write_state.argtypes = [C.c_void_p, d, d]
        L.lsm_read_state.argtypes = [C.c_void_p, d, d]
        L.lsm_read_forces.argtypes = [C.c_void_p, d]
        L.lsm_read_virial.argtypes = [C.c_void_p, d]
        L.lsm_read_strain.argtypes = [C.c_void_p, d, u8]
        L.lsm_read_broken.argtypes = [C.c_void_p, u8, i64, i64]
        L.lsm_read_energy.argtypes = [C.c_void_p, d, d]
        L.lsm_read_stress.argtypes = [C.c_void_p, C.c_int64, i64, i64, d, d, d, i64]
        L.lsm_run_to_failure.argtypes = [C.c_void_p, C.c_int64, C.c_int32, C.c_int32, C.c_double, i64, i32, d, i64]
        L.lsm_set_strain_rate.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_double, C.c_int32, C.c_int32, d]
        L.lsm_compact.argtypes = [C.c_void_p]
        L.lsm_sync.argtypes = [C.c_void_p]
        L.lsm_get_info.argtypes = [C.c_void_p, C.POINTER(LsmInfo)]
        L.lsm_device_state.argtypes = [C.c_void_p, C.POINTER(d), C.POINTER(d)]
        L.lsm_last_error.argtypes = [C.c_void_p]
        L.lsm_last_error.restype = C.c_char_p
        L.lsm_destroy.argtypes = [C.c_void_p]
        L.lsm_destroy.restype = None
        L.lsm_abi_version.restype = C.c_int32
        L.lsm_spring_energy_static.argtypes = [C.c_int32, C.c_void_p, C.c_int32, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p,
                                               C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p,
                                               C.c_char_p, C.c_size_t]
        for n in EXPORTS:
            if n not in ("lsm_last_error", "lsm_destroy", "lsm_abi_version"):
                getattr(L, n).restype = C.c_int32
        _lib = L
    return _lib


def _ptr(a, t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def _host_ptr(a, t):
    """Pointer to a host buffer: numpy array or (pinned) CPU torch tensor."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return a.ctypes.data_as(C.POINTER(t))
    return C.cast(a.data_ptr(), C.POINTER(t))      # torch CPU tensor


class _TorchAllocator:
    """Device memory from PyTorch's caching allocator, handed to the library as alloc / free callbacks."""

    def __init__(self, device):
        import torch
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.live = {}
        self.alloc_cb = _ALLOC_FN(self._alloc)
        self.free_cb = _FREE_FN(self._free)

    def _alloc(self, nbytes, _user):
        try:
            t = self.torch.empty(max(int(nbytes), 1), dtype=self.torch.uint8, device=self.device)
        except Exception:
            return None
        self.live[t.data_ptr()] = t
        return t.data_ptr()

    def _free(self, ptr, _user):
        self.live.pop(ptr, None)


class LsmSim:
    """Handle returned by lsm_create.  Methods mirror the C entry points one to one."""

    def __init__(self, handle, N, M, B, allocator, keep, D=2):
        self._h = handle
        self.N, self.M, self.B, self.D = N, M, B, D
        self._allocator = allocator
        self._keep = keep

    def _check(self, st):
        if st != 0:
            raise LsmError(st, (library().lsm_last_error(self._h) or b"").decode())

    def set_boundary(self, group, ids, mode, du=None):
        ids = np.ascontiguousarray(ids, dtype=np.int32)
        du = np.zeros(self.D) if du is None else np.ascontiguousarray(du, dtype=np.float64)
        if du.size != self.D:
            raise LsmError(-1, "disp_per_step must have dim entries")
        self._check(library().lsm_set_boundary(self._h, int(group), _ptr(ids, C.c_int32), ids.size, int(mode), _ptr(du, C.c_double)))

    def step(self, n=1):
        self._check(library().lsm_step(self._h, int(n)))

    def sync(self):
        self._check(library().lsm_sync(self._h))

    def compact(self):
        self._check(library().lsm_compact(self._h))

    def write_state(self, x, v=None):
        """x, v: [N,2] float64 host arrays (numpy or pinned torch CPU tensors)."""
        if isinstance(x, np.ndarray):
            x = np.ascontiguousarray(x, dtype=np.float64)
        if isinstance(v, np.ndarray):
            v = np.ascontiguousarray(v, dtype=np.float64)
        self._check(library().lsm_write_state(self._h, _host_ptr(x, C.c_double), _host_ptr(v, C.c_double)))

    def read_state(self, out_x=None, out_v=None):
        x = np.empty((self.N, self.D)) if out_x is None else out_x
        v = np.empty((self.N, self.D)) if out_v is None else out_v
        self._check(library().lsm_read_state(self._h, _host_ptr(x, C.c_double), _host_ptr(v, C.c_double)))
        return x, v

    def read_forces(self):
        f = np.empty((self.N, self.D))
        self._check(library().lsm_read_forces(self._h, _ptr(f, C.c_double)))
        return f

    def read_virial(self):
        S = np.empty((self.N, 3 if self.D == 2 else 6))
        self._check(library().lsm_read_virial(self._h, _ptr(S, C.c_double)))
        return S

    def read_strain(self):
        """(E [N,3] or [N,6], ok [N] bool): Lagrangian strain per particle (Eq. 8) and the full-rank flag."""
        E = np.empty((self.N, 3 if self.D == 2 else 6)); ok = np.empty(self.N, dtype=np.uint8)
        self._check(library().lsm_read_strain(self._h, _ptr(E, C.c_double), _ptr(ok, C.c_uint8)))
        return E, ok.astype(bool)

    def read_broken(self):
        b = np.empty(self.M, dtype=np.uint8); bs = np.empty(self.M, dtype=np.int64); n = C.c_int64(0)
        self._check(library().lsm_read_broken(self._h, _ptr(b, C.c_uint8), _ptr(bs, C.c_int64), C.byref(n)))
        return b.astype(bool), bs, int(n.value)

    def n_broken(self):
        n = C.c_int64(0)
        self._check(library().lsm_read_broken(self._h, None, None, C.byref(n)))
        return int(n.value)

    def read_energy(self):
        U = np.empty(self.B); KE = np.empty(self.B)
        self._check(library().lsm_read_energy(self._h, _ptr(U, C.c_double), _ptr(KE, C.c_double)))
        return U, KE

    def read_stress(self, capacity=None):
        cap = int(self.history_capacity if capacity is None else capacity)
        step = np.empty(cap, dtype=np.int64); R = np.empty((cap, self.B, MAX_GROUPS, self.D))
        U = np.empty((cap, self.B)); KE = np.empty((cap, self.B)); nb = np.empty((cap, self.B), dtype=np.int64)
        n = C.c_int64(0)
        self._check(library().lsm_read_stress(self._h, cap, C.byref(n), _ptr(step, C.c_int64), _ptr(R, C.c_double),
                                              _ptr(U, C.c_double), _ptr(KE, C.c_double), _ptr(nb, C.c_int64)))
        n = int(n.value)
        return dict(step=step[:n], R=R[:n], U=U[:n], KE=KE[:n], n_broken=nb[:n])

    def run_to_failure(self, max_steps, group=1, axis=1, stop_fraction=0.1):
        """Returns (steps_done, failed, peak[B], peak_step[B])."""
        n = C.c_int64(0); failed = C.c_int32(0)
        peak = np.zeros(self.B); pstep = np.zeros(self.B, dtype=np.int64)
        self._check(library().lsm_run_to_failure(self._h, int(max_steps), int(group), int(axis), float(stop_fraction),
                                                 C.byref(n), C.byref(failed), _ptr(peak, C.c_double), _ptr(pstep, C.c_int64)))
        return int(n.value), bool(failed.value), peak, pstep

    def set_strain_rate(self, group_lo, group_hi, axis, strain_per_step, symmetric=True, ramp=True):
        """Returns the gauge length H0."""
        h0 = C.c_double(0.0)
        self._check(library().lsm_set_strain_rate(self._h, int(group_lo), int(group_hi), int(axis), float(strain_per_step),
                                                  int(bool(symmetric)), int(bool(ramp)), C.byref(h0)))
        return float(h0.value)

    def info(self):
        inf = LsmInfo()
        self._check(library().lsm_get_info(self._h, C.byref(inf)))
        return {f[0]: getattr(inf, f[0]) for f in LsmInfo._fields_}

    @property
    def current_step(self):
        return self.info()["current_step"]

    def close(self):
        if getattr(self, "_h", None):
            library().lsm_destroy(self._h)
            self._h = None
            self._allocator = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def lsm_create(x, spring_i, spring_j, k, r0, rc, dt, gamma=0.0, v=None, mass=1.0, n_batch=1, particle_offsets=None,
               spring_offsets=None, sample_every=0, history_capacity=0, compact_every=0, reorder=REORDER_NONE,
               force_mode=FORCE_AUTO, exact=False, step_fusion=0, gather_variant=GATHER_AUTO, gather_window=0, cluster_size=0, device=0, stream=None, use_torch_allocator=True):
    """lsm_create: build a simulation from HOST arrays.  k / r0 / rc may be scalars (uniform) or [M] arrays."""
    L = library()
    x = np.ascontiguousarray(x, dtype=np.float64)
    N = int(x.shape[0])
    if x.ndim != 2:
        raise LsmError(-1, "x must be [N, dim]")
    si = np.ascontiguousarray(spring_i, dtype=np.int32)
    sj = np.ascontiguousarray(spring_j, dtype=np.int32)
    M = int(si.size)
    keep = [x, si, sj]
    d = LsmDesc()
    d.struct_size = C.sizeof(LsmDesc)
    d.dim = int(x.shape[1]); d.n_particles = N; d.n_springs = M; d.n_batch = int(n_batch)
    if particle_offsets is not None:
        po = np.ascontiguousarray(particle_offsets, dtype=np.int64); so = np.ascontiguousarray(spring_offsets, dtype=np.int64)
        keep += [po, so]
        d.particle_offsets = _ptr(po, C.c_int64); d.spring_offsets = _ptr(so, C.c_int64)
    d.x = _ptr(x, C.c_double)
    if v is not None:
        v = np.ascontiguousarray(v, dtype=np.float64); keep.append(v); d.v = _ptr(v, C.c_double)
    if np.ndim(mass) == 0:
        d.mass_uniform = float(mass)
    else:
        m = np.ascontiguousarray(mass, dtype=np.float64); keep.append(m); d.mass = _ptr(m, C.c_double)
    d.spring_i = _ptr(si, C.c_int32); d.spring_j = _ptr(sj, C.c_int32)
    for name, val in (("k", k), ("r0", r0), ("rc", rc)):
        if np.ndim(val) == 0:
            setattr(d, name + "_uniform", float(val))
        else:
            a = np.ascontiguousarray(val, dtype=np.float64)
            if a.size != M:
                raise LsmError(-1, "%s must be a scalar or have one entry per spring" % name)
            keep.append(a); setattr(d, name, _ptr(a, C.c_double))
    d.dt = float(dt); d.gamma = float(gamma)
    d.sample_every = int(sample_every); d.history_capacity = int(history_capacity); d.compact_every = int(compact_every)
    d.reorder = int(reorder); d.force_mode = int(force_mode); d.exact = int(bool(exact)); d.step_fusion = int(step_fusion)
    d.gather_variant = int(gather_variant); d.gather_window = int(gather_window); d.cluster_size = int(cluster_size)
    d.device = int(device)
    allocator = None
    try:
        import torch
        has_cuda = torch.cuda.is_available()
    except Exception:
        torch, has_cuda = None, False
    if has_cuda:
        if stream is None:
            with torch.cuda.device(device):
                stream = torch.cuda.current_stream().cuda_stream
        if use_torch_allocator:
            allocator = _TorchAllocator(device)
            d.alloc = allocator.alloc_cb; d.free_ = allocator.free_cb
    d.stream = C.c_void_p(stream or 0)
    h = C.c_void_p(None)
    st = L.lsm_create(C.byref(d), C.byref(h))
    if st != 0:
        raise LsmError(st, (L.lsm_last_error(None) or b"").decode())
    sim = LsmSim(h, N, M, int(n_batch), allocator, keep=None, D=int(x.shape[1]))
    sim.history_capacity = int(history_capacity) if history_capacity else 1024
    return sim


def lsm_create_from_problem(p, **kw):
    """Convenience: build from an lsm_inputs.Problem (arrays only) and set its boundary groups."""
    args = dict(gamma=p.gamma, v=p.v, mass=p.mass, n_batch=p.n_batch, particle_offsets=p.particle_offsets,
                spring_offsets=p.spring_offsets, sample_every=p.sample_every)
    args.update(kw)
    sim = lsm_create(p.x, p.spring_i, p.spring_j, p.k, p.r0, p.rc, p.dt, **args)
    for gi, g in enumerate(p.groups):
        sim.set_boundary(gi, g.ids, g.mode, g.du)
    return sim


# ---- free-function spellings of the C names ----
def lsm_set_boundary(sim, group, ids, mode, du=None): return sim.set_boundary(group, ids, mode, du)
def lsm_step(sim, n=1): return sim.step(n)
def lsm_write_state(sim, x, v=None): return sim.write_state(x, v)
def lsm_read_state(sim, out_x=None, out_v=None): return sim.read_state(out_x, out_v)
def lsm_read_forces(sim): return sim.read_forces()
def lsm_read_virial(sim): return sim.read_virial()
def lsm_read_strain(sim): return sim.read_strain()
def lsm_read_broken(sim): return sim.read_broken()
def lsm_read_energy(sim): return sim.read_energy()
def lsm_read_stress(sim, capacity=None): return sim.read_stress(capacity)
def lsm_run_to_failure(sim, max_steps, group=1, axis=1, stop_fraction=0.1): return sim.run_to_failure(max_steps, group, axis, stop_fraction)
def lsm_set_strain_rate(sim, group_lo, group_hi, axis, strain_per_step, symmetric=True, ramp=True): return sim.set_strain_rate(group_lo, group_hi, axis, strain_per_step, symmetric, ramp)
def lsm_compact(sim): return sim.compact()
def lsm_sync(sim): return sim.sync()
def lsm_get_info(sim): return sim.info()
def lsm_destroy(sim): return sim.close()
def lsm_last_error(sim=None): return (library().lsm_last_error(sim._h if sim is not None else None) or b"").decode()
def lsm_abi_version(): return int(library().lsm_abi_version())


def lsm_spring_energy_static(x, spring_i, spring_j, k, r0, U, broken=None, counts=None, stream=None):
    """lsm_spring_energy_static: elastic energy (Eq. 1) of a spring list that already sits on the GPU, for callers that
    cannot allocate there (see include/lsm.h for who they are).  Marshalling only, and in keeping with the entry point
    this wrapper creates no tensor either: every array is a CUDA tensor the caller made earlier -- x [N, dim] float64,
    spring_i / spring_j [M] int32, k / r0 [M] float64 or Python scalars (uniform), broken [M] uint8 or None, U [1] float64
    (output), counts [2] int64 or None (output: springs summed, springs skipped for bad ids).  Contiguous tensors on one
    device; the work is enqueued on `stream` (default: torch's current stream on that device) and U is valid once that
    stream has been synchronised.  Raises LsmError(-2) for more than STATIC_MAX_SPRINGS springs."""
    import torch
    dev = x.device.index if x.device.index is not None else torch.cuda.current_device()

    def dptr(t, dtype, n, name):
        if t is None:
            return None
        if not (t.is_cuda and t.device.index == dev and t.dtype == dtype and t.is_contiguous() and t.numel() == n):
            raise LsmError(-1, "%s must be a contiguous %s CUDA tensor with %d entries on device %d" % (name, dtype, n, dev))
        return C.c_void_p(t.data_ptr())

    if x.dim() != 2:
        raise LsmError(-1, "x must be [N, dim]")
    N, D, M = int(x.shape[0]), int(x.shape[1]), int(spring_i.numel())
    k_t, k_u = (None, float(k)) if not hasattr(k, "data_ptr") else (k, 0.0)
    r0_t, r0_u = (None, float(r0)) if not hasattr(r0, "data_ptr") else (r0, 0.0)
    if stream is None:
        stream = torch.cuda.current_stream(dev).cuda_stream
    err = C.create_string_buffer(512)
    st = library().lsm_spring_energy_static(
        dev, C.c_void_p(stream or 0), D, N, M, dptr(x, torch.float64, N * D, "x"), dptr(spring_i, torch.int32, M, "spring_i"),
        dptr(spring_j, torch.int32, M, "spring_j"), dptr(k_t, torch.float64, M, "k"), dptr(r0_t, torch.float64, M, "r0"), k_u, r0_u,
        dptr(broken, torch.uint8, M, "broken"), dptr(U, torch.float64, 1, "U"), dptr(counts, torch.int64, 2, "counts"), err, len(err))
    if st != 0:
        raise LsmError(st, err.value.decode())

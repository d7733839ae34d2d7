"""Thin ctypes binding over the C-ABI library (include/glisse.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; this module holds no arithmetic of the
method and has no CPU fallback: if libglisse.so is missing and cannot be built with nvcc, or no
CUDA device is usable, it raises.  Names follow the C ABI: GlisseSim.create/advance/read ...

Host inputs are numpy float64 arrays; device inputs are torch CUDA float64 tensors (PyTorch is
used for device memory and streams only).
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_double, c_int, c_longlong, c_void_p

import numpy as np

from . import build as _build

OK, EINVAL, ECUDA, ENOMEM, EPLANET, ELIMIT = 0, -1, -2, -3, -4, -5
FLAG_ACTIVE, FLAG_RMIN, FLAG_RMAX, FLAG_NONCONV, FLAG_UNBOUND, FLAG_PLANET0 = 0, 1, 2, 3, 4, 16

#: every symbol include/glisse.h declares (tests check that the library exports each one) ...
EXPORTS = (
    "glisse_default_params", "glisse_create", "glisse_advance", "glisse_advance_with_log", "glisse_set_planets",
    "glisse_log_stride", "glisse_planet_log", "glisse_planet_log_static", "glisse_planet_log_static_limit",
    "glisse_interpolate_log", "glisse_read", "glisse_read_planets",
    "glisse_snapshot", "glisse_snapshot_wait", "glisse_snapshot_ring", "glisse_snapshots_emitted",
    "glisse_resonance_begin", "glisse_resonance_sample", "glisse_resonance_read", "glisse_libration_read",
    "glisse_active_count", "glisse_step", "glisse_particle_steps", "glisse_sync", "glisse_destroy", "glisse_run",
    "glisse_strerror",
)
#: ... and the measurement / test hooks of include/glisse_test.h
TEST_EXPORTS = (
    "glisse_launch_count", "glisse_particle_kernel_time", "glisse_fp64_peak_probe", "glisse_test_primitive",
    "glisse_solver_stats_enable", "glisse_solver_stats",
)


class GlisseParams(ctypes.Structure):
    _fields_ = [("r_min", c_double), ("r_max", c_double), ("kepler_iters", c_int), ("kepler_tol", c_double),
                ("chunk_steps", c_int), ("resync_chunks", c_int), ("device", c_int), ("stream", c_void_p),
                ("snapshot_chunks", c_int), ("resonance_chunks", c_int), ("bin_iterations", c_int),
                ("scheme", c_int), ("guess_order", c_int), ("segment_steps", c_int)]


class GlisseError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__(f"{where}: {strerror(status)} (status {status})")


_lib = None


def library_path() -> str:
    return _build.LIB


def lib():
    """Load libglisse.so (building it in-tree with nvcc if it is missing or stale)."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        P3 = POINTER(c_void_p)
        L.glisse_default_params.argtypes = [POINTER(GlisseParams)]
        L.glisse_default_params.restype = None
        L.glisse_create.argtypes = [POINTER(c_void_p), c_double, c_int, c_void_p, c_void_p, c_void_p, c_void_p,
                                    c_longlong, P3, P3, c_double, POINTER(GlisseParams)]
        L.glisse_create.restype = c_int
        L.glisse_advance.argtypes = [c_void_p, c_longlong]
        L.glisse_advance.restype = c_int
        L.glisse_advance_with_log.argtypes = [c_void_p, c_longlong, c_void_p]
        L.glisse_advance_with_log.restype = c_int
        L.glisse_set_planets.argtypes = [c_void_p, c_void_p, c_void_p]
        L.glisse_set_planets.restype = c_int
        L.glisse_snapshot_ring.argtypes = [c_void_p, c_int, c_int, c_void_p, c_void_p, c_void_p, c_void_p]
        L.glisse_snapshot_ring.restype = c_int
        L.glisse_snapshots_emitted.argtypes = [c_void_p]
        L.glisse_snapshots_emitted.restype = c_longlong
        L.glisse_libration_read.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]
        L.glisse_libration_read.restype = c_int
        L.glisse_solver_stats_enable.argtypes = [c_void_p, c_int]
        L.glisse_solver_stats_enable.restype = c_int
        L.glisse_solver_stats.argtypes = [c_void_p, POINTER(c_longlong), POINTER(c_longlong), POINTER(c_longlong)]
        L.glisse_solver_stats.restype = c_int
        L.glisse_log_stride.argtypes = [c_int]
        L.glisse_log_stride.restype = c_int
        L.glisse_planet_log.argtypes = [c_void_p, c_longlong, c_void_p]
        L.glisse_planet_log.restype = c_int
        L.glisse_planet_log_static.argtypes = [c_void_p, c_longlong, c_void_p]
        L.glisse_planet_log_static.restype = c_int
        L.glisse_planet_log_static_limit.argtypes = [c_int]
        L.glisse_planet_log_static_limit.restype = c_longlong
        L.glisse_interpolate_log.argtypes = [c_void_p, c_longlong, c_void_p, c_void_p, c_void_p, c_double, c_double,
                                             c_longlong, c_void_p]
        L.glisse_interpolate_log.restype = c_int
        L.glisse_read.argtypes = [c_void_p, P3, P3, c_void_p, c_void_p]
        L.glisse_read.restype = c_int
        L.glisse_snapshot.argtypes = [c_void_p, c_int, POINTER(c_void_p), c_void_p, c_void_p]
        L.glisse_snapshot.restype = c_int
        L.glisse_snapshot_wait.argtypes = [c_void_p]
        L.glisse_snapshot_wait.restype = c_int
        L.glisse_resonance_begin.argtypes = [c_void_p, c_int, c_int, c_int, c_double]
        L.glisse_resonance_begin.restype = c_int
        L.glisse_resonance_sample.argtypes = [c_void_p]
        L.glisse_resonance_sample.restype = c_int
        L.glisse_resonance_read.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, POINTER(c_longlong)]
        L.glisse_resonance_read.restype = c_int
        L.glisse_read_planets.argtypes = [c_void_p, c_void_p, c_void_p]
        L.glisse_read_planets.restype = c_int
        for name in ("glisse_active_count", "glisse_step", "glisse_particle_steps", "glisse_launch_count"):
            getattr(L, name).argtypes = [c_void_p]
            getattr(L, name).restype = c_longlong
        L.glisse_sync.argtypes = [c_void_p]
        L.glisse_sync.restype = c_int
        L.glisse_particle_kernel_time.argtypes = [c_void_p, POINTER(c_double), POINTER(c_longlong)]
        L.glisse_particle_kernel_time.restype = c_int
        L.glisse_fp64_peak_probe.argtypes = [c_int, c_void_p, c_double, POINTER(c_double)]
        L.glisse_fp64_peak_probe.restype = c_int
        L.glisse_test_primitive.argtypes = [c_int, c_longlong, c_void_p, c_void_p]
        L.glisse_test_primitive.restype = c_int
        L.glisse_destroy.argtypes = [c_void_p]
        L.glisse_destroy.restype = None
        L.glisse_run.argtypes = [c_double, c_int, c_void_p, c_void_p, c_void_p, c_void_p, c_longlong, P3, P3, c_double,
                                 POINTER(GlisseParams), c_longlong, c_int, P3, P3, c_void_p, c_void_p,
                                 POINTER(c_longlong)]
        L.glisse_run.restype = c_int
        L.glisse_strerror.argtypes = [c_int]
        L.glisse_strerror.restype = ctypes.c_char_p
        _lib = L
    return _lib


def strerror(status: int) -> str:
    return lib().glisse_strerror(int(status)).decode()


def planet_log_static_limit(n_planets: int) -> int:
    return int(lib().glisse_planet_log_static_limit(int(n_planets)))


def log_stride(n_planets: int) -> int:
    return lib().glisse_log_stride(int(n_planets))


def _check(status, where):
    if status != OK:
        raise GlisseError(status, where)


def _is_torch(t) -> bool:
    return type(t).__module__.startswith("torch")


def _ptr(a):
    """Raw address of a numpy array or torch tensor (None -> NULL)."""
    if a is None:
        return None
    if _is_torch(a):
        return c_void_p(a.data_ptr())
    return c_void_p(a.ctypes.data)


def _rows(a, n_rows):
    """Three (or n_rows) contiguous float64 rows of a [n_rows, N] numpy array or torch tensor."""
    if _is_torch(a):
        import torch
        assert a.dtype == torch.float64 and a.shape[0] == n_rows
        a = a.contiguous()
        return a, [a[k] for k in range(n_rows)]
    a = np.ascontiguousarray(a, dtype=np.float64)
    assert a.shape[0] == n_rows
    return a, [a[k] for k in range(n_rows)]


def _p3(rows):
    return (c_void_p * 3)(*[(r.data_ptr() if _is_torch(r) else r.ctypes.data) for r in rows])


def _params(*, r_min=0.0, r_max=float("inf"), kepler_iters=5, kepler_tol=1e-14, chunk_steps=1024, resync_chunks=1,
            device=0, stream=None, snapshot_chunks=0, resonance_chunks=0, bin_iterations=2, segment_steps=None,
            scheme="kdk", guess_order=0):
    """glisse_params from keywords (defaults = glisse_default_params)."""
    prm = GlisseParams()
    lib().glisse_default_params(byref(prm))
    prm.r_min, prm.r_max = float(r_min), float(r_max)
    prm.kepler_iters, prm.kepler_tol = int(kepler_iters), float(kepler_tol)
    prm.chunk_steps, prm.resync_chunks = int(chunk_steps), int(resync_chunks)
    prm.device = int(device)
    prm.stream = None if stream is None else c_void_p(int(stream))
    prm.snapshot_chunks, prm.resonance_chunks = int(snapshot_chunks), int(resonance_chunks)
    prm.bin_iterations = int(bin_iterations)
    prm.scheme = {"kdk": 0, "dkd": 1}[scheme]
    prm.guess_order = int(guess_order)
    if segment_steps is not None:
        prm.segment_steps = int(segment_steps)
    return prm


def run(w, n_steps, n_parts=0, out=None, **kw):
    """glisse_run on a workload (inputs.Workload fields): create + advance(n_steps) + read + destroy, pipelined
    over n_parts slices of the particles (0 = automatic).  w.pos / w.vel: [3, N] numpy arrays (pinned for the
    copies to overlap) or torch CUDA tensors; out = (pos[3,N], vel[3,N], flag[N] int32, removal_step[N] int64)
    or None (allocated, pageable).  Returns (pos, vel, flag, removal_step, particle_steps)."""
    kw.setdefault("chunk_steps", w.chunk_steps)
    prm = _params(r_min=w.r_min, r_max=w.r_max, **kw)
    gm_planet = np.ascontiguousarray(w.gm_planet, dtype=np.float64).reshape(-1)
    npl = int(gm_planet.shape[0])
    ppos = np.ascontiguousarray(w.planet_pos, dtype=np.float64).reshape(npl, 3)
    pvel = np.ascontiguousarray(w.planet_vel, dtype=np.float64).reshape(npl, 3)
    rcrit = None if w.planet_rcrit is None else np.ascontiguousarray(w.planet_rcrit, dtype=np.float64).reshape(npl)
    keep_p, prow = _rows(w.pos, 3)
    keep_v, vrow = _rows(w.vel, 3)
    n = int(prow[0].shape[0])
    if out is None:
        out = (np.empty((3, n), dtype=np.float64), np.empty((3, n), dtype=np.float64),
               np.empty(n, dtype=np.int32), np.empty(n, dtype=np.int64))
    pos, vel, flag, rstep = out
    ps = c_longlong(0)
    st = lib().glisse_run(float(w.gm_star), npl, _ptr(gm_planet), _ptr(ppos), _ptr(pvel), _ptr(rcrit), n, _p3(prow),
                          _p3(vrow), float(w.dt), byref(prm), int(n_steps), int(n_parts),
                          None if pos is None else _p3([pos[k] for k in range(3)]),
                          None if vel is None else _p3([vel[k] for k in range(3)]), _ptr(flag), _ptr(rstep),
                          byref(ps))
    _check(st, "glisse_run")
    return pos, vel, flag, rstep, int(ps.value)


class GlisseSim:
    """glisse_create / glisse_advance / glisse_read with the C ABI's argument order."""

    def __init__(self, gm_star, gm_planet, planet_pos, planet_vel, planet_rcrit, pos, vel, dt, *, r_min=0.0,
                 r_max=float("inf"), kepler_iters=5, kepler_tol=1e-14, chunk_steps=1024, resync_chunks=1,
                 device=0, stream=None, snapshot_chunks=0, resonance_chunks=0, bin_iterations=2,
                 segment_steps=None, scheme="kdk", guess_order=0):
        L = lib()
        gm_planet = np.ascontiguousarray(gm_planet, dtype=np.float64).reshape(-1)
        self.n_planets = int(gm_planet.shape[0])
        planet_pos = np.ascontiguousarray(planet_pos, dtype=np.float64).reshape(self.n_planets, 3)
        planet_vel = np.ascontiguousarray(planet_vel, dtype=np.float64).reshape(self.n_planets, 3)
        rcrit = None if planet_rcrit is None else np.ascontiguousarray(planet_rcrit, dtype=np.float64).reshape(
            self.n_planets)
        keep_p, prow = _rows(pos, 3)
        keep_v, vrow = _rows(vel, 3)
        self.n = int(prow[0].shape[0])
        self.device = int(device)
        prm = _params(r_min=r_min, r_max=r_max, kepler_iters=kepler_iters, kepler_tol=kepler_tol,
                      chunk_steps=chunk_steps, resync_chunks=resync_chunks, device=device, stream=stream,
                      snapshot_chunks=snapshot_chunks, resonance_chunks=resonance_chunks,
                      bin_iterations=bin_iterations, segment_steps=segment_steps, scheme=scheme,
                      guess_order=guess_order)
        h = c_void_p()
        st = L.glisse_create(byref(h), float(gm_star), self.n_planets, _ptr(gm_planet), _ptr(planet_pos),
                             _ptr(planet_vel), _ptr(rcrit), self.n, _p3(prow), _p3(vrow), float(dt), byref(prm))
        self._h = None
        _check(st, "glisse_create")
        self._h = h

    @classmethod
    def from_workload(cls, w, **kw):
        kw.setdefault("chunk_steps", w.chunk_steps)
        return cls(w.gm_star, w.gm_planet, w.planet_pos, w.planet_vel, w.planet_rcrit, w.pos, w.vel, w.dt,
                   r_min=w.r_min, r_max=w.r_max, **kw)

    # ---- the calls of include/glisse.h ---------------------------------------------------------
    def advance(self, n_steps):
        _check(lib().glisse_advance(self._h, int(n_steps)), "glisse_advance")

    def advance_with_log(self, n_steps, log):
        if not _is_torch(log):
            log = np.ascontiguousarray(log, dtype=np.float64)
        assert log.shape[0] >= n_steps + 1
        _check(lib().glisse_advance_with_log(self._h, int(n_steps), _ptr(log)), "glisse_advance_with_log")

    def set_planets(self, planet_pos, planet_vel):
        pp = np.ascontiguousarray(planet_pos, dtype=np.float64).reshape(self.n_planets, 3)
        pv = np.ascontiguousarray(planet_vel, dtype=np.float64).reshape(self.n_planets, 3)
        _check(lib().glisse_set_planets(self._h, _ptr(pp), _ptr(pv)), "glisse_set_planets")

    def planet_log(self, n_steps):
        out = np.zeros((int(n_steps) + 1, log_stride(self.n_planets)), dtype=np.float64)
        _check(lib().glisse_planet_log(self._h, int(n_steps), _ptr(out)), "glisse_planet_log")
        return out

    def planet_log_static(self, n_steps, out):
        """glisse_planet_log_static: the same log written straight into `out`, a torch CUDA float64 tensor
        [n_steps + 1, stride] the caller allocated; the library allocates nothing."""
        _check(lib().glisse_planet_log_static(self._h, int(n_steps), _ptr(out)), "glisse_planet_log_static")
        return out

    def interpolate_log(self, sample_time, sample_pos, sample_vel, t_first, dt_record, n_records, out=None):
        """Planet log [n_records, stride] interpolated from a sparse history: sample_time [M], sample_pos /
        sample_vel [M, Np, 3] (numpy or torch CUDA float64); out: optional numpy / torch CUDA buffer."""
        if out is None:
            out = np.empty((int(n_records), log_stride(self.n_planets)), dtype=np.float64)
        keep = []
        def as_arg(t):
            if _is_torch(t):
                t = t.contiguous(); keep.append(t); return t
            t = np.ascontiguousarray(t, dtype=np.float64); keep.append(t); return t
        st, sq, sv = as_arg(sample_time), as_arg(sample_pos), as_arg(sample_vel)
        n_samples = int(st.shape[0])
        _check(lib().glisse_interpolate_log(self._h, n_samples, _ptr(st), _ptr(sq), _ptr(sv), float(t_first),
                                            float(dt_record), int(n_records), _ptr(out)), "glisse_interpolate_log")
        return out

    def read(self, out=None):
        """Returns (pos[3,N], vel[3,N], flag[N] int32, removal_step[N] int64) as host numpy arrays,
        or fills the given (pos, vel, flag, removal_step) numpy arrays / torch CUDA tensors."""
        if out is None:
            pos = np.empty((3, self.n), dtype=np.float64)
            vel = np.empty((3, self.n), dtype=np.float64)
            flag = np.empty(self.n, dtype=np.int32)
            rstep = np.empty(self.n, dtype=np.int64)
        else:
            pos, vel, flag, rstep = out
        prow = None if pos is None else [pos[k] for k in range(3)]
        vrow = None if vel is None else [vel[k] for k in range(3)]
        st = lib().glisse_read(self._h, None if prow is None else _p3(prow), None if vrow is None else _p3(vrow),
                               _ptr(flag), _ptr(rstep))
        _check(st, "glisse_read")
        return pos, vel, flag, rstep

    def snapshot(self, kind="cartesian", out=None):
        """glisse_snapshot: queue an asynchronous copy of the state at the current step and return
        at once.  kind: "cartesian" (x, y, z, vx, vy, vz) or "elements" (a, e, i, Omega, omega, M).
        out = (data[6,N], flag[N] int32, removal_step[N] int64): numpy arrays (pinned, e.g. views of
        pinned torch tensors, for the copy to overlap) or torch CUDA tensors; allocated (pageable)
        when omitted.  The arrays are valid after snapshot_wait()."""
        k = {"cartesian": 0, "elements": 1}[kind]
        if out is None:
            data = np.empty((6, self.n), dtype=np.float64)
            flag = np.empty(self.n, dtype=np.int32)
            rstep = np.empty(self.n, dtype=np.int64)
        else:
            data, flag, rstep = out
        rows = None
        if data is not None:
            rows = (c_void_p * 6)(*[(data[j].data_ptr() if _is_torch(data) else data[j].ctypes.data)
                                    for j in range(6)])
        st = lib().glisse_snapshot(self._h, k, rows, _ptr(flag), _ptr(rstep))
        _check(st, "glisse_snapshot")
        self._snap_keep = (data, flag, rstep)   # keep the buffers alive until the wait
        return data, flag, rstep

    def snapshot_wait(self):
        _check(lib().glisse_snapshot_wait(self._h), "glisse_snapshot_wait")
        self._snap_keep = None

    def snapshot_ring(self, kind, n_slots, data=None, flag=None, removal_step=None, slot_step=None):
        """glisse_snapshot_ring: attach the output ring of the periodic snapshots (params
        snapshot_chunks).  data [n_slots, 6, N] float64 (+ optional flag [n_slots, N] int32, removal_step
        [n_slots, N] int64, slot_step [n_slots] int64): numpy (pinned) or torch CUDA; allocated
        (pageable numpy) when data is None.  Returns the arrays; they are kept alive by the sim."""
        k = {"cartesian": 0, "elements": 1}[kind]
        if data is None and n_slots > 0:
            data = np.empty((n_slots, 6, self.n), dtype=np.float64)
            flag = np.empty((n_slots, self.n), dtype=np.int32)
            removal_step = np.empty((n_slots, self.n), dtype=np.int64)
            slot_step = np.full(n_slots, -1, dtype=np.int64)
        _check(lib().glisse_snapshot_ring(self._h, k, int(n_slots), _ptr(data), _ptr(flag), _ptr(removal_step),
                                          _ptr(slot_step)), "glisse_snapshot_ring")
        self._ring_keep = (data, flag, removal_step, slot_step)
        return data, flag, removal_step, slot_step

    def snapshots_emitted(self):
        return self._count(lib().glisse_snapshots_emitted, "glisse_snapshots_emitted")

    def libration_read(self):
        """(phi_min[N], phi_max[N], amp_mean[N], amp_max[N], n_amp[N] int32)"""
        lo = np.empty(self.n, dtype=np.float64)
        hi = np.empty(self.n, dtype=np.float64)
        mean = np.empty(self.n, dtype=np.float64)
        amax = np.empty(self.n, dtype=np.float64)
        cnt = np.empty(self.n, dtype=np.int32)
        _check(lib().glisse_libration_read(self._h, _ptr(lo), _ptr(hi), _ptr(mean), _ptr(amax), _ptr(cnt)),
               "glisse_libration_read")
        return lo, hi, mean, amax, cnt

    def solver_stats_enable(self, on=True):
        _check(lib().glisse_solver_stats_enable(self._h, 1 if on else 0), "glisse_solver_stats_enable")

    def solver_stats(self):
        """(warp drift calls, fast-solver iterations summed over them, calls that entered the slow path)"""
        a, b, c = c_longlong(), c_longlong(), c_longlong()
        _check(lib().glisse_solver_stats(self._h, byref(a), byref(b), byref(c)), "glisse_solver_stats")
        return a.value, b.value, c.value

    def resonance_begin(self, planet, p, q, window):
        _check(lib().glisse_resonance_begin(self._h, int(planet), int(p), int(q), float(window)),
               "glisse_resonance_begin")

    def resonance_sample(self):
        _check(lib().glisse_resonance_sample(self._h), "glisse_resonance_sample")

    def resonance_read(self):
        """(seen0[N] uint8, seen180[N] uint8, phi_last[N], n_samples)"""
        s0 = np.empty(self.n, dtype=np.uint8)
        s180 = np.empty(self.n, dtype=np.uint8)
        phi = np.empty(self.n, dtype=np.float64)
        ns = c_longlong(0)
        _check(lib().glisse_resonance_read(self._h, _ptr(s0), _ptr(s180), _ptr(phi), byref(ns)),
               "glisse_resonance_read")
        return s0, s180, phi, int(ns.value)

    def read_planets(self):
        pos = np.empty((self.n_planets, 3), dtype=np.float64)
        vel = np.empty((self.n_planets, 3), dtype=np.float64)
        _check(lib().glisse_read_planets(self._h, _ptr(pos), _ptr(vel)), "glisse_read_planets")
        return pos, vel

    def _count(self, fn, where):
        v = int(fn(self._h))
        if v < 0:
            raise GlisseError(v, where)
        return v

    def active_count(self):
        return self._count(lib().glisse_active_count, "glisse_active_count")

    def step(self):
        return self._count(lib().glisse_step, "glisse_step")

    def particle_steps(self):
        return self._count(lib().glisse_particle_steps, "glisse_particle_steps")

    def launch_count(self):
        return self._count(lib().glisse_launch_count, "glisse_launch_count")

    def sync(self):
        _check(lib().glisse_sync(self._h), "glisse_sync")

    def particle_kernel_time(self):
        """(milliseconds, launches) spent in particle kernels since the last call."""
        ms, n = c_double(), c_longlong()
        _check(lib().glisse_particle_kernel_time(self._h, byref(ms), byref(n)), "glisse_particle_kernel_time")
        return ms.value, n.value

    def close(self):
        if getattr(self, "_h", None):
            lib().glisse_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def fp64_peak_probe(device=0, millis=200.0, stream=None) -> float:
    """Measured FP64 FMA rate of the device in FLOP/s (register-resident DFMA loop)."""
    out = c_double()
    st = lib().glisse_fp64_peak_probe(int(device), None if stream is None else c_void_p(int(stream)), float(millis),
                                      byref(out))
    _check(st, "glisse_fp64_peak_probe")
    return out.value


_PRIM = {"rsqrt": (0, 1, 1), "rcp": (1, 1, 1), "rcp1": (2, 1, 1), "sincosm": (3, 1, 2), "kepler_drift": (4, 10, 7),
         "kepler_drift_refined": (5, 10, 7)}


def test_primitive(name, x):
    """Evaluate one device primitive on a host array (test hook of include/glisse.h)."""
    which, n_in, n_out = _PRIM[name]
    x = np.ascontiguousarray(x, dtype=np.float64)
    n = x.size // n_in
    out = np.empty(n * n_out, dtype=np.float64)
    _check(lib().glisse_test_primitive(which, n, _ptr(x), _ptr(out)), "glisse_test_primitive")
    return out.reshape(n, n_out) if n_out > 1 else out


test_primitive.__test__ = False  # not a pytest test

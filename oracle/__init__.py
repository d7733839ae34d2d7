"""ctypes loader for the ORACLE (oracle/glisse_oracle.cpp).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / `--impl reference` legs.  Nothing under paper_2011_03484_b200/ imports this
package and this package imports nothing from there.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import POINTER, c_double, c_int, c_longlong, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "glisse_oracle.cpp")
_LIB = os.path.join(_HERE, "libglisse_oracle.so")

#: no FMA contraction, plain libm; -O2 only so the arithmetic is what the source says
CXXFLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-Wall"]


def build(force: bool = False) -> str:
    """Compile the oracle with g++ if the shared object is missing or older than the source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.run(["g++", *CXXFLAGS, _SRC, "-o", tmp, "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


class _Params(ctypes.Structure):
    _fields_ = [("r_min", c_double), ("r_max", c_double), ("kepler_iters", c_int),
                ("kepler_tol", c_double), ("scheme", c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        P3 = POINTER(c_void_p)
        L.oracle_create.argtypes = [POINTER(c_void_p), c_double, c_int, c_void_p, c_void_p, c_void_p,
                                    c_void_p, c_longlong, P3, P3, c_double, POINTER(_Params)]
        L.oracle_create.restype = c_int
        for name in ("oracle_advance",):
            getattr(L, name).argtypes = [c_void_p, c_longlong]
            getattr(L, name).restype = c_int
        L.oracle_planet_log.argtypes = [c_void_p, c_longlong, c_void_p]
        L.oracle_planet_log.restype = c_int
        L.oracle_interpolate_log.argtypes = [c_int, c_void_p, c_longlong, c_void_p, c_void_p, c_void_p, c_double,
                                             c_double, c_longlong, c_void_p]
        L.oracle_interpolate_log.restype = c_int
        L.oracle_advance_with_log.argtypes = [c_void_p, c_longlong, c_void_p]
        L.oracle_advance_with_log.restype = c_int
        L.oracle_read.argtypes = [c_void_p, P3, P3, c_void_p, c_void_p]
        L.oracle_read.restype = c_int
        L.oracle_read_planets.argtypes = [c_void_p, c_void_p, c_void_p]
        L.oracle_read_planets.restype = c_int
        for name in ("oracle_active_count", "oracle_step", "oracle_particle_steps"):
            getattr(L, name).argtypes = [c_void_p]
            getattr(L, name).restype = c_longlong
        L.oracle_destroy.argtypes = [c_void_p]
        L.oracle_destroy.restype = None
        L.oracle_log_stride.argtypes = [c_int]
        L.oracle_log_stride.restype = c_int
        L.oracle_default_params.argtypes = [POINTER(_Params)]
        L.oracle_elements.argtypes = [c_double, c_void_p, c_void_p, c_void_p]
        L.oracle_elements.restype = None
        L.oracle_resonant_argument.argtypes = [c_double, c_void_p, c_void_p, c_double, c_void_p, c_void_p,
                                               c_int, c_int]
        L.oracle_resonant_argument.restype = c_double
        L.oracle_libration_summary.argtypes = [c_void_p, c_longlong, c_double, c_void_p]
        L.oracle_libration_summary.restype = None
        L.oracle_kepler_drift.argtypes = [c_double, c_void_p, c_void_p, c_double, c_int, c_double]
        L.oracle_kepler_drift.restype = c_int
        L.oracle_planet_kick_accel.argtypes = [c_int, c_double, c_void_p, c_void_p, c_void_p]
        L.oracle_planet_kick_accel.restype = c_int
        L.oracle_helio_to_jacobi.argtypes = [c_int, c_double, c_void_p, c_void_p, c_void_p]
        L.oracle_jacobi_to_helio.argtypes = [c_int, c_double, c_void_p, c_void_p, c_void_p]
        L.oracle_planet_step.argtypes = [c_int, c_double, c_void_p, c_void_p, c_void_p, c_double]
        L.oracle_planet_step.restype = c_int
        L.oracle_particle_accel.argtypes = [c_int, c_void_p, c_void_p, c_void_p, c_double, c_double,
                                            c_void_p, c_void_p]
        L.oracle_particle_accel.restype = c_int
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(c_void_p)


def _p3(arrs):
    return (c_void_p * 3)(*[a.ctypes.data for a in arrs])


class OracleSim:
    """Same call sequence as the CUDA binding's GlisseSim: create / advance / read."""

    def __init__(self, gm_star, gm_planet, planet_pos, planet_vel, planet_rcrit, pos, vel, dt,
                 r_min=0.0, r_max=float("inf"), kepler_iters=5, kepler_tol=1e-14, scheme="kdk"):
        L = lib()
        gm_planet = _f64(gm_planet).reshape(-1)
        self.np_ = int(gm_planet.shape[0])
        planet_pos = _f64(planet_pos).reshape(self.np_, 3)
        planet_vel = _f64(planet_vel).reshape(self.np_, 3)
        rcrit = None if planet_rcrit is None else _f64(planet_rcrit).reshape(self.np_)
        pos = _f64(pos)
        vel = _f64(vel)
        assert pos.shape == vel.shape and pos.shape[0] == 3
        self.n = int(pos.shape[1])
        prm = _Params(float(r_min), float(r_max), int(kepler_iters), float(kepler_tol),
                      {"kdk": 0, "dkd": 1}[scheme])
        h = c_void_p()
        xs = [np.ascontiguousarray(pos[k]) for k in range(3)]
        vs = [np.ascontiguousarray(vel[k]) for k in range(3)]
        st = L.oracle_create(ctypes.byref(h), float(gm_star), self.np_, _p(gm_planet), _p(planet_pos),
                             _p(planet_vel), None if rcrit is None else _p(rcrit), self.n, _p3(xs),
                             _p3(vs), float(dt), ctypes.byref(prm))
        if st != 0:
            raise ValueError(f"oracle_create failed with status {st}")
        self._h = h

    @classmethod
    def from_workload(cls, w, **kw):
        return cls(w.gm_star, w.gm_planet, w.planet_pos, w.planet_vel, w.planet_rcrit, w.pos, w.vel,
                   w.dt, r_min=w.r_min, r_max=w.r_max, **kw)

    def advance(self, n_steps):
        st = lib().oracle_advance(self._h, int(n_steps))
        if st != 0:
            raise RuntimeError(f"oracle_advance failed with status {st}")

    def log_stride(self):
        return lib().oracle_log_stride(self.np_)

    def planet_log(self, n_steps):
        out = np.zeros((int(n_steps) + 1, self.log_stride()), dtype=np.float64)
        st = lib().oracle_planet_log(self._h, int(n_steps), _p(out))
        if st != 0:
            raise RuntimeError(f"oracle_planet_log failed with status {st}")
        return out

    def advance_with_log(self, n_steps, log):
        log = _f64(log)
        assert log.shape[0] >= n_steps + 1
        st = lib().oracle_advance_with_log(self._h, int(n_steps), _p(log))
        if st != 0:
            raise RuntimeError(f"oracle_advance_with_log failed with status {st}")

    def read(self):
        pos = np.empty((3, self.n), dtype=np.float64)
        vel = np.empty((3, self.n), dtype=np.float64)
        flag = np.empty(self.n, dtype=np.int32)
        rstep = np.empty(self.n, dtype=np.int64)
        st = lib().oracle_read(self._h, _p3([pos[k] for k in range(3)]), _p3([vel[k] for k in range(3)]),
                               _p(flag), _p(rstep))
        assert st == 0
        return pos, vel, flag, rstep

    def read_planets(self):
        pos = np.empty((self.np_, 3), dtype=np.float64)
        vel = np.empty((self.np_, 3), dtype=np.float64)
        assert lib().oracle_read_planets(self._h, _p(pos), _p(vel)) == 0
        return pos, vel

    def active_count(self):
        return int(lib().oracle_active_count(self._h))

    def step(self):
        return int(lib().oracle_step(self._h))

    def particle_steps(self):
        return int(lib().oracle_particle_steps(self._h))

    def close(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- single-function entry points for the pins -------------------------------------------------

def elements(mu, pos, vel):
    """Osculating elements (a, e, i, Omega, omega, M) of each column of pos, vel ([3, N]) -> [6, N]."""
    L = lib()
    pos = np.ascontiguousarray(np.asarray(pos, dtype=np.float64).T)
    vel = np.ascontiguousarray(np.asarray(vel, dtype=np.float64).T)
    out = np.empty((pos.shape[0], 6))
    for k in range(pos.shape[0]):
        L.oracle_elements(c_double(mu), _p(pos[k]), _p(vel[k]), _p(out[k]))
    return np.ascontiguousarray(out.T)


def resonant_argument(mu, pos, vel, mu_pl, rp, vp, p, q):
    """phi = p lambda − q lambda_pl − (p − q) varpi of each column of pos, vel ([3, N]) -> [N]."""
    L = lib()
    pos = np.ascontiguousarray(np.asarray(pos, dtype=np.float64).T)
    vel = np.ascontiguousarray(np.asarray(vel, dtype=np.float64).T)
    rp, vp = _f64(rp), _f64(vp)
    return np.array([L.oracle_resonant_argument(c_double(mu), _p(pos[k]), _p(vel[k]), c_double(mu_pl), _p(rp),
                                                _p(vp), int(p), int(q)) for k in range(pos.shape[0])])


def libration_summary(phi, window):
    """Libration summary of sampled resonant arguments.  phi: [n_samples] or [n_samples, N] (time along
    axis 0) -> dict of seen0, seen180 (bool), phi_min, phi_max, amp_mean, amp_max, n_amp per particle."""
    L = lib()
    phi = np.asarray(phi, dtype=np.float64)
    one = phi.ndim == 1
    series = np.ascontiguousarray(phi.reshape(phi.shape[0], -1).T)     # [N, n_samples]
    out = np.empty((series.shape[0], 7))
    for k in range(series.shape[0]):
        L.oracle_libration_summary(_p(series[k]), series.shape[1], c_double(window), _p(out[k]))
    d = dict(seen0=out[:, 0] != 0, seen180=out[:, 1] != 0, phi_min=out[:, 2], phi_max=out[:, 3],
             amp_mean=out[:, 4], amp_max=out[:, 5], n_amp=out[:, 6].astype(np.int64))
    return {k: v[0] for k, v in d.items()} if one else d


def interpolate_log(gm_planet, sample_time, sample_pos, sample_vel, t_first, dt_record, n_records):
    """Planet log [n_records, stride] by cubic Hermite interpolation of a sparse history:
    sample_time [M], sample_pos / sample_vel [M, Np, 3] heliocentric."""
    gm = _f64(gm_planet).reshape(-1)
    npl = gm.shape[0]
    t = _f64(sample_time).reshape(-1)
    q = _f64(sample_pos).reshape(t.shape[0], npl, 3)
    v = _f64(sample_vel).reshape(t.shape[0], npl, 3)
    stride = lib().oracle_log_stride(npl)
    out = np.zeros((int(n_records), stride), dtype=np.float64)
    st = lib().oracle_interpolate_log(npl, _p(gm), t.shape[0], _p(t), _p(q), _p(v), float(t_first), float(dt_record),
                                      int(n_records), _p(out))
    if st != 0:
        raise ValueError(f"oracle_interpolate_log refused its arguments (status {st})")
    return out


def kepler_drift(mu, r, v, dt, iters=5, tol=1e-14):
    """O2 on one body. Returns (flag, r_new, v_new)."""
    r = _f64(r).copy()
    v = _f64(v).copy()
    fl = lib().oracle_kepler_drift(float(mu), _p(r), _p(v), float(dt), int(iters), float(tol))
    return fl, r, v


def planet_kick_accel(gm0, gm, q):
    gm = _f64(gm)
    q = _f64(q)
    acc = np.zeros_like(q)
    assert lib().oracle_planet_kick_accel(len(gm), float(gm0), _p(gm), _p(q), _p(acc)) == 0
    return acc


def helio_to_jacobi(gm0, gm, h):
    gm = _f64(gm)
    h = _f64(h)
    out = np.zeros_like(h)
    lib().oracle_helio_to_jacobi(len(gm), float(gm0), _p(gm), _p(h), _p(out))
    return out


def jacobi_to_helio(gm0, gm, j):
    gm = _f64(gm)
    j = _f64(j)
    out = np.zeros_like(j)
    lib().oracle_jacobi_to_helio(len(gm), float(gm0), _p(gm), _p(j), _p(out))
    return out


def planet_step(gm0, gm, q, qd, dt):
    gm = _f64(gm)
    q = _f64(q).copy()
    qd = _f64(qd).copy()
    st = lib().oracle_planet_step(len(gm), float(gm0), _p(gm), _p(q), _p(qd), float(dt))
    return st, q, qd


def particle_accel(gm, q, rcrit, r_min, r_max, r):
    gm = _f64(gm)
    q = _f64(q)
    r = _f64(r)
    a = np.zeros(3)
    rc = None if rcrit is None else _f64(rcrit)
    fl = lib().oracle_particle_accel(len(gm), _p(gm), _p(q), None if rc is None else _p(rc),
                                     float(r_min), float(r_max), _p(r), _p(a))
    return fl, a

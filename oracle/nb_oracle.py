"""ctypes front-end of the CPU oracle (oracle/nb_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It never
imports the CUDA package and the CUDA package never imports it.

Every function cites the passage of PAPER.md it restates in nb_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nb_oracle.c")
_LIB = os.path.join(_HERE, "libnb_oracle.so")
_lib = None

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_lp = C.POINTER(C.c_int64)


def build(force: bool = False) -> str:
    """Compile nb_oracle.c with gcc (plain C11, OpenMP, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-std=c11", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def build_plain_double(force: bool = False) -> str:
    """The same source with the arithmetic type set to double and -O3 -march=native: bench.py's
    plain-double CPU throughput baseline (never used as a correctness reference)."""
    out = os.path.join(_HERE, "libnb_oracle_f64.so")
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-std=c11", "-O3", "-march=native", "-fopenmp", "-ffp-contract=off", "-DORC_REAL=double",
               "-DORC_SQRT=sqrt", "-fPIC", "-shared", "-o", out, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return out


def force_plain_double_rate(pos_pred, vel_pred, acc_pred, mass, eps, idx):
    """Pairs/s of orc_force in the plain-double build on the rows idx (timing aid for bench.py)."""
    import time
    L = C.CDLL(build_plain_double())
    L.orc_force.argtypes = [C.c_int64, _dp, _dp, _dp, _dp, C.c_double, _ip, C.c_int64, _dp, _dp, _dp]
    rp, vp, ap, m = _arr(pos_pred), _arr(vel_pred), _arr(acc_pred), _arr(mass)
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    n = idx.shape[0]
    acc = np.zeros((n, 3)); jerk = np.zeros((n, 3)); snap = np.zeros((n, 3))
    t0 = time.perf_counter()
    L.orc_force(m.shape[0], _d(rp), _d(vp), _d(ap), _d(m), float(eps), idx.ctypes.data_as(_ip), n, _d(acc), _d(jerk), _d(snap))
    return n * m.shape[0] / (time.perf_counter() - t0), acc


def _d(x):
    return x.ctypes.data_as(_dp)


def _arr(x, shape=None):
    a = np.ascontiguousarray(x, dtype=np.float64)
    if shape is not None:
        a = a.reshape(shape)
    return a


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_force.argtypes = [C.c_int64, _dp, _dp, _dp, _dp, C.c_double, _ip, C.c_int64, _dp, _dp, _dp]
        L.orc_force_mixed.argtypes = [C.c_int64, _dp, _dp, _dp, _dp, C.c_double, _ip, C.c_int64, _dp, _dp, _dp, _dp]
        L.orc_predict.argtypes = [C.c_int64, C.c_double] + [_dp] * 10
        L.orc_correct_particle.argtypes = [C.c_double] + [_dp] * 13
        L.orc_timestep.argtypes = [_dp] * 6 + [C.c_double] * 5
        L.orc_timestep.restype = C.c_double
        L.orc_initial_dt.argtypes = [_dp] * 3 + [C.c_double] * 3
        L.orc_initial_dt.restype = C.c_double
        L.orc_energy.argtypes = [C.c_int64, _dp, _dp, _dp, C.c_double, _dp]
        L.orc_create.argtypes = [C.c_int64, _dp, _dp, _dp, C.c_double, C.c_double]
        L.orc_create.restype = C.c_void_p
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_limits.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double]
        L.orc_startup.argtypes = [C.c_void_p]
        L.orc_next_block.argtypes = [C.c_void_p]
        L.orc_next_block.restype = C.c_double
        L.orc_step.argtypes = [C.c_void_p]
        L.orc_run_until.argtypes = [C.c_void_p, C.c_double, _dp, _lp, C.c_int64]
        L.orc_run_until.restype = C.c_int64
        for name in ("mass", "t", "dt", "pos", "vel", "acc", "jerk", "snap", "crackle",
                     "pos_pred", "vel_pred", "acc_pred"):
            getattr(L, "orc_get_" + name).argtypes = [C.c_void_p, _dp]
        L.orc_t_now.argtypes = [C.c_void_p]; L.orc_t_now.restype = C.c_double
        L.orc_t_next.argtypes = [C.c_void_p]; L.orc_t_next.restype = C.c_double
        L.orc_n_active.argtypes = [C.c_void_p]; L.orc_n_active.restype = C.c_int64
        L.orc_get_active.argtypes = [C.c_void_p, _ip]
        L.orc_n_steps.argtypes = [C.c_void_p]; L.orc_n_steps.restype = C.c_int64
        L.orc_n_pairs.argtypes = [C.c_void_p]; L.orc_n_pairs.restype = C.c_double
        L.orc_get_hist.argtypes = [C.c_void_p, _lp]
        L.orc_state_energy.argtypes = [C.c_void_p, _dp]
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(int(n))


def force(pos_pred, vel_pred, acc_pred, mass, eps, idx=None):
    """Eq. 8-10 with Eq. 2 softening: (acc, jerk, snap), each [n_idx, 3]."""
    rp, vp, ap = _arr(pos_pred), _arr(vel_pred), _arr(acc_pred)
    m = _arr(mass)
    N = m.shape[0]
    if idx is None:
        n, ip = N, None
    else:
        idx = np.ascontiguousarray(idx, dtype=np.int32)
        n, ip = idx.shape[0], idx.ctypes.data_as(_ip)
    acc = np.zeros((n, 3)); jerk = np.zeros((n, 3)); snap = np.zeros((n, 3))
    lib().orc_force(N, _d(rp), _d(vp), _d(ap), _d(m), float(eps), ip, n, _d(acc), _d(jerk), _d(snap))
    return acc, jerk, snap


def force_mixed(pos_pred, vel_pred, acc_pred, mass, eps, idx=None):
    """Eq. 8-10 in the paper's mixed precision (reading G27): DP differences, SP pair
    arithmetic.  Returns (acc, jerk, snap, scale), scale[k] = sum_j |pair term|_2 per quantity."""
    rp, vp, ap = _arr(pos_pred), _arr(vel_pred), _arr(acc_pred)
    m = _arr(mass)
    N = m.shape[0]
    if idx is None:
        n, ip = N, None
    else:
        idx = np.ascontiguousarray(idx, dtype=np.int32)
        n, ip = idx.shape[0], idx.ctypes.data_as(_ip)
    acc = np.zeros((n, 3)); jerk = np.zeros((n, 3)); snap = np.zeros((n, 3)); scale = np.zeros((n, 3))
    lib().orc_force_mixed(N, _d(rp), _d(vp), _d(ap), _d(m), float(eps), ip, n, _d(acc), _d(jerk), _d(snap), _d(scale))
    return acc, jerk, snap, scale


def predict(t, ti, r, v, a, j, s, c):
    """Eq. 3-7: (r_pred, v_pred, a_pred) at time t, interval t - t_i."""
    ti = _arr(ti); N = ti.shape[0]
    ins = [_arr(x, (N, 3)) for x in (r, v, a, j, s, c)]
    rp = np.zeros((N, 3)); vp = np.zeros((N, 3)); ap = np.zeros((N, 3))
    lib().orc_predict(N, float(t), _d(ti), *[_d(x) for x in ins], _d(rp), _d(vp), _d(ap))
    return rp, vp, ap


def correct_particle(h, r0, v0, a0, j0, s0, a1, j1, s1):
    """Eq. 11-14 + end-point a^(3), a^(4), a^(5): (r1, v1, c3, c4, c5)."""
    ins = [_arr(x, (3,)) for x in (r0, v0, a0, j0, s0, a1, j1, s1)]
    outs = [np.zeros(3) for _ in range(5)]
    lib().orc_correct_particle(float(h), *[_d(x) for x in ins], *[_d(x) for x in outs])
    return tuple(outs)


def timestep(a, j, s, c3, c4, c5, eta, dt_old, t_next, dt_min, dt_max):
    """Eq. 15-16, p = 6, power-of-two quantisation."""
    ins = [_arr(x, (3,)) for x in (a, j, s, c3, c4, c5)]
    return float(lib().orc_timestep(*[_d(x) for x in ins], float(eta), float(dt_old), float(t_next),
                                    float(dt_min), float(dt_max)))


def initial_dt(a, j, s, eta_init, dt_min, dt_max):
    ins = [_arr(x, (3,)) for x in (a, j, s)]
    return float(lib().orc_initial_dt(*[_d(x) for x in ins], float(eta_init), float(dt_min), float(dt_max)))


def energy(pos, vel, mass, eps):
    """Eq. 2 / Eq. 20: array [E, K, W, Px, Py, Pz, Lx, Ly, Lz]."""
    r, v, m = _arr(pos), _arr(vel), _arr(mass)
    out = np.zeros(9)
    lib().orc_energy(m.shape[0], _d(r), _d(v), _d(m), float(eps), _d(out))
    return out


class Integrator:
    """The Hermite 6th-order block-time-step loop of PAPER.md:54-102 (oracle state)."""

    def __init__(self, pos, vel, mass, eps, eta, dt_min=2.0 ** -25, dt_max=2.0 ** -3, eta_init=0.01,
                 startup=True):
        r, v, m = _arr(pos), _arr(vel), _arr(mass)
        self.N = m.shape[0]
        self._L = lib()
        self._h = C.c_void_p(self._L.orc_create(self.N, _d(r), _d(v), _d(m), float(eps), float(eta)))
        self._L.orc_set_limits(self._h, float(dt_min), float(dt_max), float(eta_init))
        if startup:
            self._L.orc_startup(self._h)

    def __del__(self):
        try:
            self._L.orc_destroy(self._h)
        except Exception:
            pass

    def _get(self, name, shape):
        out = np.zeros(shape)
        getattr(self._L, "orc_get_" + name)(self._h, _d(out))
        return out

    pos = property(lambda s: s._get("pos", (s.N, 3)))
    vel = property(lambda s: s._get("vel", (s.N, 3)))
    acc = property(lambda s: s._get("acc", (s.N, 3)))
    jerk = property(lambda s: s._get("jerk", (s.N, 3)))
    snap = property(lambda s: s._get("snap", (s.N, 3)))
    crackle = property(lambda s: s._get("crackle", (s.N, 3)))
    pos_pred = property(lambda s: s._get("pos_pred", (s.N, 3)))
    vel_pred = property(lambda s: s._get("vel_pred", (s.N, 3)))
    acc_pred = property(lambda s: s._get("acc_pred", (s.N, 3)))
    mass = property(lambda s: s._get("mass", (s.N,)))
    t = property(lambda s: s._get("t", (s.N,)))
    dt = property(lambda s: s._get("dt", (s.N,)))
    t_now = property(lambda s: float(s._L.orc_t_now(s._h)))
    n_steps = property(lambda s: int(s._L.orc_n_steps(s._h)))
    n_pairs = property(lambda s: float(s._L.orc_n_pairs(s._h)))

    def next_block(self):
        """Table 1 row 1: (t_next, ascending active indices)."""
        tn = float(self._L.orc_next_block(self._h))
        m = int(self._L.orc_n_active(self._h))
        act = np.zeros(m, dtype=np.int32)
        self._L.orc_get_active(self._h, act.ctypes.data_as(_ip))
        return tn, act

    def step(self):
        self._L.orc_step(self._h)

    def run_until(self, t_end, log_cap=0):
        lt = np.zeros(max(log_cap, 1)); lm = np.zeros(max(log_cap, 1), dtype=np.int64)
        n = int(self._L.orc_run_until(self._h, float(t_end), _d(lt), lm.ctypes.data_as(_lp), int(log_cap)))
        k = min(n, log_cap)
        return n, lt[:k], lm[:k]

    def hist(self):
        h = np.zeros(64, dtype=np.int64)
        self._L.orc_get_hist(self._h, h.ctypes.data_as(_lp))
        return h

    def energy(self):
        out = np.zeros(9)
        self._L.orc_state_energy(self._h, _d(out))
        return out

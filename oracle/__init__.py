"""ctypes loader for the parity oracle (oracle/aw_oracle.cpp) — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports the CUDA package and shares no code with it.  Arrays are numpy,
SoA planes exactly as DESIGN.md §4 lays them out (q[6, pitch], w[6, pitch], acc[4, pitch],
wind[3, pitch], status[n]); the arithmetic all lives in the C++ file, this module only marshals.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "aw_oracle.cpp")
_LIB = os.path.join(_HERE, "libaw_oracle.so")
_FLAGS = ["-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared"]

_lib = None


def build(force=False):
    """Compile oracle/aw_oracle.cpp -> oracle/libaw_oracle.so (g++, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["g++"] + _FLAGS + ["-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


class Grid(C.Structure):
    _fields_ = [("gx", C.c_int32), ("gy", C.c_int32),
                ("lo_x", C.c_double), ("hi_x", C.c_double), ("lo_y", C.c_double), ("hi_y", C.c_double),
                ("angle_mode", C.c_int32), ("shape", C.c_int32),
                ("cx", C.c_double), ("cy", C.c_double), ("r", C.c_double),
                ("pz_sign", C.c_int32), ("tangent_mode", C.c_int32), ("k0", C.c_int64),
                ("resample", C.c_int32), ("reserved_", C.c_int32)]


def make_grid(gx, gy, lo=-1.0, hi=1.0, angle_mode=0, shape=0, cx=0.0, cy=0.0, r=0.0, pz_sign=1,
              tangent_mode=0, lo_y=None, hi_y=None, k0=0, resample=0):
    """The grid describes the WHOLE ensemble (gx*gy trajectories); a State of n trajectories initialised
    with it holds the slice [k0, k0 + n)."""
    return Grid(gx, gy, lo, hi, lo if lo_y is None else lo_y, hi if hi_y is None else hi_y,
                angle_mode, shape, cx, cy, r, pz_sign, tangent_mode, k0, resample, 0)


_dp = C.POINTER(C.c_double)
_i32p = C.POINTER(C.c_int32)
_u8p = C.POINTER(C.c_uint8)
_u32p = C.POINTER(C.c_uint32)
_u64p = C.POINTER(C.c_uint64)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.awo_hp.restype = C.c_double
        L.awo_hp.argtypes = [C.c_double] * 3
        L.awo_grad.argtypes = [C.c_double] * 3 + [_dp]
        L.awo_hess.argtypes = [C.c_double] * 3 + [_dp]
        L.awo_hamiltonian.restype = C.c_double
        L.awo_hamiltonian.argtypes = [_dp, C.c_double]
        L.awo_stage_list.argtypes = [C.c_int, _dp]
        L.awo_stage_constants.argtypes = [C.c_int, C.c_double, C.c_double, _dp, _dp]
        L.awo_mix64.restype = C.c_uint64
        L.awo_mix64.argtypes = [C.c_uint64, C.c_uint64]
        L.awo_uniform.restype = C.c_double
        L.awo_uniform.argtypes = [C.c_uint64] * 3
        L.awo_common_tangent.argtypes = [C.c_uint64, _dp]
        L.awo_steps.argtypes = [_dp, _dp, C.c_int, C.c_double, C.c_double, C.c_int64]
        L.awo_checkpoint.argtypes = [_dp, _dp, _dp, _i32p, C.c_double, _dp]
        L.awo_init_shell.argtypes = [C.POINTER(Grid), C.c_double, C.c_double, C.c_uint64, C.c_int64,
                                     C.c_int64, _dp, _dp, _dp, _i32p, _u8p]
        L.awo_integrate.argtypes = [C.c_int64, C.c_int64, _dp, _dp, _dp, _i32p, _u8p, C.c_double,
                                    C.c_int, C.c_int64, C.c_double, C.c_int64, C.c_int64, C.c_int64, _dp]
        L.awo_indicator.argtypes = [C.c_int64, C.c_int64, _dp, _u8p, C.c_double, C.c_int, C.c_double,
                                    _dp, _u8p]
        L.awo_density.argtypes = [C.c_int64, C.c_int64, _dp, _u8p, _u32p, C.c_int32, C.c_int32,
                                  C.c_double, C.c_double, _u64p]
        L.awo_mark.argtypes = [C.c_int64, _dp, _i32p, _dp, _i32p]
        L.awo_velocity.argtypes = [C.c_int64, C.c_int64, _dp, _i32p, _dp, _i32p, _u8p, C.c_double, C.c_double,
                                   C.c_int, _dp]
        L.awo_density_velocity.argtypes = [C.c_int64, C.c_int64, _dp, _i32p, _dp, _i32p, _u8p, C.c_double,
                                           C.c_double, C.c_int, _u32p, C.c_int32, C.c_int32, C.c_double,
                                           C.c_double, _u64p]
        L.awo_delta_p.argtypes = [C.c_int64, C.c_int64, _dp, _dp, _u8p, _dp]
        L.awo_energy_stats.argtypes = [C.c_int64, C.c_int64, _dp, _dp, _u8p, C.c_double, _dp, _dp]
        _lib = L
    return _lib


def _p(a, t):
    return None if a is None else a.ctypes.data_as(t)


# ----------------------------------------------------------------------------- scalar helpers

def hp(x, y, z):
    return lib().awo_hp(x, y, z)


def grad(x, y, z):
    g = np.zeros(3)
    lib().awo_grad(x, y, z, _p(g, _dp))
    return g


def hess(x, y, z):
    h = np.zeros(9)
    lib().awo_hess(x, y, z, _p(h, _dp))
    return h.reshape(3, 3)


def hamiltonian(q, eps):
    q = np.ascontiguousarray(q, dtype=np.float64)
    return lib().awo_hamiltonian(_p(q, _dp), eps)


def stage_list(order):
    w = np.zeros(9)
    S = lib().awo_stage_list(order, _p(w, _dp))
    return w[:S].copy()


def stage_constants(order, dt, eps):
    a, b = np.zeros(10), np.zeros(9)
    S = lib().awo_stage_constants(order, dt, eps, _p(a, _dp), _p(b, _dp))
    return a[:S + 1].copy(), b[:S].copy()


def mix64(seed, ctr):
    return lib().awo_mix64(seed, ctr)


def uniform(seed, k, slot):
    return lib().awo_uniform(seed, k, slot)


def common_tangent(seed):
    t = np.zeros(6)
    lib().awo_common_tangent(seed, _p(t, _dp))
    return t


def steps(q, tw, order, dt, eps, nsteps):
    """`nsteps` plain steps (no checkpoint / wrap) on one trajectory; returns new (q, tw)."""
    q = np.array(q, dtype=np.float64)
    tw = None if tw is None else np.array(tw, dtype=np.float64)
    rc = lib().awo_steps(_p(q, _dp), _p(tw, _dp), order, dt, eps, nsteps)
    assert rc == 0
    return q, tw


def checkpoint(q, tw, acc, wind, eps, surv=None):
    q = np.array(q, dtype=np.float64)
    tw = None if tw is None else np.array(tw, dtype=np.float64)
    acc = np.array(acc, dtype=np.float64)
    wind = None if wind is None else np.array(wind, dtype=np.int32)
    surv = None if surv is None else np.array(surv, dtype=np.float64)
    st = lib().awo_checkpoint(_p(q, _dp), _p(tw, _dp), _p(acc, _dp), _p(wind, _i32p), eps, _p(surv, _dp))
    return q, tw, acc, wind, st


# ----------------------------------------------------------------------------- ensemble state

class State:
    """SoA ensemble state on the host (numpy), mirroring the planes of aw_state."""

    def __init__(self, n, tangent=True, wind=True, pitch=None):
        self.n = int(n)
        self.pitch = int(pitch) if pitch else (self.n + 31) // 32 * 32
        self.q = np.zeros((6, self.pitch))
        self.w = np.zeros((6, self.pitch)) if tangent else None
        self.acc = np.zeros((4, self.pitch))
        self.wind = np.zeros((3, self.pitch), dtype=np.int32) if wind else None
        self.status = np.zeros(self.n, dtype=np.uint8)
        self.E = float("nan")
        self.eps = float("nan")
        self.t = 0.0
        self.step = 0
        self.order = 4
        self.qref = None        # snapshot taken by mark(): start of the averaging window
        self.windref = None
        self.tref = 0.0
        self.surv = None        # survivor rectangle (lo_x, hi_x, lo_y, hi_y) or None

    def copy(self):
        s = State(self.n, self.w is not None, self.wind is not None, self.pitch)
        s.q[:] = self.q
        if self.w is not None:
            s.w[:] = self.w
        s.acc[:] = self.acc
        if self.wind is not None:
            s.wind[:] = self.wind
        s.status[:] = self.status
        s.E, s.eps, s.t, s.step, s.order = self.E, self.eps, self.t, self.step, self.order
        s.qref = None if self.qref is None else self.qref.copy()
        s.windref = None if self.windref is None else self.windref.copy()
        s.tref, s.surv = self.tref, self.surv
        return s


def init_shell(state, grid, E, eps, seed):
    rc = lib().awo_init_shell(C.byref(grid), E, eps, seed, state.n, state.pitch, _p(state.q, _dp),
                              _p(state.w, _dp), _p(state.acc, _dp), _p(state.wind, _i32p),
                              _p(state.status, _u8p))
    assert rc == 0, rc
    state.E, state.eps, state.t, state.step = E, eps, 0.0, 0
    return state


def integrate(state, steps, dt, stride, k0=0, k1=None, advance_clock=True):
    """Integrate trajectories [k0, k1) (default all).  Single-threaded; callers may run disjoint
    ranges from several Python threads (ctypes drops the GIL) — the arithmetic is per trajectory."""
    k1 = state.n if k1 is None else k1
    surv = None if state.surv is None else np.array(state.surv, dtype=np.float64)
    rc = lib().awo_integrate(state.n, state.pitch, _p(state.q, _dp), _p(state.w, _dp),
                             _p(state.acc, _dp), _p(state.wind, _i32p), _p(state.status, _u8p),
                             state.eps, state.order, steps, dt, stride, k0, k1, _p(surv, _dp))
    assert rc == 0, rc
    if advance_clock:
        state.t += steps * abs(dt)
        state.step += steps
    return state


def indicator(state, kind, thr=0.0):
    if kind == 3:
        out = np.zeros(state.n, dtype=np.uint8)
        rc = lib().awo_indicator(state.n, state.pitch, _p(state.acc, _dp), _p(state.status, _u8p),
                                 state.t, kind, thr, None, _p(out, _u8p))
    else:
        out = np.zeros(state.n)
        rc = lib().awo_indicator(state.n, state.pitch, _p(state.acc, _dp), _p(state.status, _u8p),
                                 state.t, kind, thr, _p(out, _dp), None)
    assert rc == 0, rc
    return out


def density(state, hist, lo, hi, dropped=None):
    """Add the live trajectories' (px, py) into hist[gy, gx] (uint32, C order); returns dropped."""
    gy, gx = hist.shape
    d = np.zeros(1, dtype=np.uint64) if dropped is None else dropped
    rc = lib().awo_density(state.n, state.pitch, _p(state.q, _dp), _p(state.status, _u8p),
                           _p(hist, _u32p), gx, gy, lo, hi, _p(d, _u64p))
    assert rc == 0, rc
    return d


def mark(state):
    """Snapshot (q, wind) as the start of an averaging window / the reference P(0) of P:37."""
    state.qref = np.zeros_like(state.q)
    state.windref = None if state.wind is None else np.zeros_like(state.wind)
    rc = lib().awo_mark(state.pitch, _p(state.q, _dp), _p(state.wind, _i32p), _p(state.qref, _dp),
                        _p(state.windref, _i32p))
    assert rc == 0, rc
    state.tref = state.t
    return state


def velocity(state, projected=True):
    """[3, n] averaged finite-time velocity over [tref, t], centrally projected on S if asked."""
    out = np.zeros((3, state.n))
    rc = lib().awo_velocity(state.n, state.pitch, _p(state.q, _dp), _p(state.wind, _i32p),
                            _p(state.qref, _dp), _p(state.windref, _i32p), _p(state.status, _u8p),
                            state.E, state.t - state.tref, 1 if projected else 0, _p(out, _dp))
    assert rc == 0, rc
    return out


def density_velocity(state, hist, lo, hi, hemi=1, dropped=None):
    """Add the projected averaged velocities (Vhat_x, Vhat_y) of one hemisphere (1: z >= 0, 2: z < 0,
    3: both) into hist[gy, gx]; returns dropped."""
    gy, gx = hist.shape
    d = np.zeros(1, dtype=np.uint64) if dropped is None else dropped
    rc = lib().awo_density_velocity(state.n, state.pitch, _p(state.q, _dp), _p(state.wind, _i32p),
                                    _p(state.qref, _dp), _p(state.windref, _i32p), _p(state.status, _u8p),
                                    state.E, state.t - state.tref, hemi, _p(hist, _u32p), gx, gy, lo, hi,
                                    _p(d, _u64p))
    assert rc == 0, rc
    return d


def delta_p(state):
    """||P(t) - P(tref)|| per trajectory."""
    out = np.zeros(state.n)
    rc = lib().awo_delta_p(state.n, state.pitch, _p(state.q, _dp), _p(state.qref, _dp),
                           _p(state.status, _u8p), _p(out, _dp))
    assert rc == 0, rc
    return out


def energy_stats(state):
    """(stats[8], signed dH image[n]) — the energy-drift statistics of BASELINE configs[2] (R29)."""
    out, img = np.zeros(8), np.zeros(state.n)
    rc = lib().awo_energy_stats(state.n, state.pitch, _p(state.q, _dp), _p(state.acc, _dp),
                                _p(state.status, _u8p), state.eps, _p(out, _dp), _p(img, _dp))
    assert rc == 0, rc
    return out, img

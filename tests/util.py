"""Test-side helpers: move a device ensemble into an oracle State, run the oracle on all host cores."""
import math
import os
import threading

import numpy as np

TWO_PI = 2.0 * math.pi


def ensemble_to_oracle(ens, orc):
    """Copy the device planes of a paper_1107_4107_b200.Ensemble into a fresh oracle.State (R11: for
    parity runs the GPU-generated initial conditions are handed to the oracle)."""
    st = orc.State(ens.n, tangent=ens.w is not None, wind=ens.wind is not None, pitch=ens.pitch)
    st.q[:] = ens.q.cpu().numpy()
    if ens.w is not None:
        st.w[:] = ens.w.cpu().numpy()
    st.acc[:] = ens.acc.cpu().numpy()
    if ens.wind is not None:
        st.wind[:] = ens.wind.cpu().numpy()
    st.status[:] = ens.status[:ens.n].cpu().numpy()
    st.E, st.eps, st.t, st.step, st.order = ens.E, ens.eps, ens.t, ens.step, ens.order
    if getattr(ens, "qref", None) is not None:           # snapshot of aw_mark (window start)
        st.qref = ens.qref.cpu().numpy().copy()
        st.windref = None if ens.windref is None else ens.windref.cpu().numpy().copy()
        st.tref = ens.tref
    if ens.c.survive:
        st.surv = (ens.c.surv_lo_x, ens.c.surv_hi_x, ens.c.surv_lo_y, ens.c.surv_hi_y)
    return st


def oracle_integrate_mt(orc, st, steps, dt, stride, subset=None, threads=None):
    """Run oracle.integrate over disjoint trajectory ranges on all host cores (the arithmetic is per
    trajectory, ctypes drops the GIL).  subset: iterable of (k0, k1) ranges, default the whole ensemble."""
    threads = threads or os.cpu_count() or 1
    ranges = []
    if subset is None:
        edges = np.linspace(0, st.n, threads + 1).astype(np.int64)
        ranges = [(int(a), int(b)) for a, b in zip(edges[:-1], edges[1:]) if b > a]
    else:
        ranges = list(subset)
    pending = list(ranges)
    lock = threading.Lock()

    def work():
        while True:
            with lock:
                if not pending:
                    return
                k0, k1 = pending.pop()
            orc.integrate(st, steps, dt, stride, k0=k0, k1=k1, advance_clock=False)

    ts = [threading.Thread(target=work) for _ in range(min(threads, len(ranges)))]
    [t.start() for t in ts]
    [t.join() for t in ts]
    st.t += steps * abs(dt)
    st.step += steps
    return st


def unwrapped(q, wind):
    """angles + 2 pi * turns (compare across wraps)."""
    out = q.copy()
    if wind is not None:
        out[:3] = out[:3] + TWO_PI * wind
    return out


def state_rel_err(q_gpu, wind_gpu, q_ref, wind_ref, live):
    """Per-trajectory relative error of the state, angles and actions normalised SEPARATELY:
    max(|dX|_inf / max(1, |X|_inf), |dP|_inf / max(1, |P|_inf)) with X the unwrapped angles, so that a large
    unwrapped angle cannot loosen the bar on the momenta (BASELINE north_star: "state within 1e-10 relative")."""
    a = unwrapped(q_gpu, wind_gpu)[:, live]
    b = unwrapped(q_ref, wind_ref)[:, live]
    d = np.abs(a - b)
    sx = np.maximum(1.0, np.max(np.abs(b[:3]), axis=0))
    sp = np.maximum(1.0, np.max(np.abs(b[3:]), axis=0))
    return np.maximum(np.max(d[:3], axis=0) / sx, np.max(d[3:], axis=0) / sp)


def load_oracle_variant(name, extra_flags, out_dir):
    """A second, separately built copy of the oracle (same source, extra compiler flags) as its own module
    object: used by the rounding experiment (-include tests/jitter_trig.h) and the sanitizer build."""
    import importlib.util
    import oracle
    spec = importlib.util.spec_from_file_location("oracle_" + name, oracle.__file__)
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    m._LIB = os.path.join(str(out_dir), "libaw_oracle_%s.so" % name)
    m._FLAGS = list(m._FLAGS) + list(extra_flags)
    m.build(force=True)
    return m

"""The host oracle under -fsanitize=address,undefined (sanitizer row): the oracle's own source rebuilt
with both sanitizers and driven through pins P1 (free motion), P5 (reversibility) and P12 (histogram brute force and
edges), plus the generator with every shape, slices and resampling, in a subprocess with the sanitizer runtime
preloaded (an instrumented shared object cannot be loaded into an uninstrumented python otherwise).  Any report —
out-of-bounds plane access, misaligned load, signed overflow, invalid shift, float-to-int overflow — fails the test.
compute-sanitizer is closed on the GPU pool, so this is the sanitizer evidence available."""
import os
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = textwrap.dedent('''
    import math, sys
    import numpy as np
    sys.path.insert(0, %(root)r); sys.path.insert(0, %(tests)r)
    from util import load_oracle_variant
    orc = load_oracle_variant("asan", ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-g",
                                       "-fno-omit-frame-pointer"], %(out)r)
    # P1: eps = 0, closed form (P:35)
    for order in (4, 6):
        st = orc.init_shell(orc.State(33), orc.make_grid(33, 1, angle_mode=1, tangent_mode=1), 1.0, 0.0, 5)
        st.order = order
        q0 = st.q.copy()
        orc.integrate(st, 700, 0.01, 100)
        assert np.array_equal(st.q[3:], q0[3:])
        X = st.q[:3] + 2 * math.pi * st.wind
        assert np.max(np.abs(X - (q0[:3] + 7.0 * q0[3:]))) < 1e-11
    # P5: forward then backward (north_star: within 1e-12)
    st = orc.init_shell(orc.State(64, tangent=True), orc.make_grid(8, 8, angle_mode=1), 1.0, 1e-2, 0)
    q0 = st.q.copy()
    orc.integrate(st, 1000, 0.01, 100)
    orc.integrate(st, 1000, -0.01, 100)
    X = st.q[:3] + 2 * math.pi * st.wind
    live = st.status == 1
    assert np.max(np.abs(X - q0[:3])[:, :64][:, live]) < 1e-11 and np.max(np.abs(st.q[3:] - q0[3:])[:, :64][:, live]) < 1e-12
    # P12: histogram vs numpy, bin edges, ragged n, dropped points; velocity density, dP, energy statistics
    n = 1003
    st = orc.State(n, tangent=False)
    rng = np.random.default_rng(12)
    st.q[3, :n] = rng.uniform(-1.2, 1.2, n); st.q[4, :n] = rng.uniform(-1.2, 1.2, n)
    st.q[3, :6] = [-1.0, 1.0, 1.0 - 2 ** -53, -0.0, np.nan, np.inf]
    st.status[:] = 1; st.status[::17] = 0
    for G, lo, hi in ((64, -1.0, 1.0), (1, -1.0, 1.0), (255, -0.5, 0.7)):
        h = np.zeros((G, G), dtype=np.uint32)
        d = orc.density(st, h, lo, hi)
        assert int(h.sum()) + int(d[0]) == int((st.status == 1).sum())
    st.E, st.eps = 1.0, 1e-2
    orc.mark(st)
    st.t = 3.0
    st.q[:3, :n] += rng.uniform(-1, 1, (3, n)); st.wind[:, :n] += rng.integers(-3, 4, (3, n)).astype(np.int32)
    hv = np.zeros((32, 32), dtype=np.uint32)
    for hemi in (1, 2, 3):
        orc.density_velocity(st, hv, -1.5, 1.5, hemi)
    orc.velocity(st); orc.delta_p(st); orc.energy_stats(st)
    for kind in (0, 1, 2, 3):
        orc.indicator(st, kind, 1.0)
    # generator: every shape, a slice, resampling, survivor filter
    for shape in (0, 1, 2, 3):
        g = orc.make_grid(13, 7, -0.9, 0.9, 1, shape, 0.99, 0.98, 0.05, -1, 1, k0=20, resample=3)
        s2 = orc.init_shell(orc.State(60), g, 1.0, 3e-2, 9)
        s2.surv = (-0.5, 0.5, -0.5, 0.5)
        orc.integrate(s2, 200, 0.005, 100)
    print("SANITIZED-OK")
''')


def _runtime(name):
    p = subprocess.run(["gcc", "-print-file-name=" + name], capture_output=True, text=True).stdout.strip()
    return p if os.path.isabs(p) and os.path.exists(p) else None


def test_oracle_runs_clean_under_asan_and_ubsan(tmp_path):
    asan, ubsan = _runtime("libasan.so"), _runtime("libubsan.so")
    if not asan or not ubsan:
        pytest.skip("gcc sanitizer runtimes not installed")
    env = dict(os.environ, LD_PRELOAD=asan + ":" + ubsan,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:exitcode=66", UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    code = DRIVER % dict(root=ROOT, tests=os.path.join(ROOT, "tests"), out=str(tmp_path))
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, env=env, timeout=600)
    report = r.stdout[-3000:] + r.stderr[-6000:]
    assert r.returncode == 0, report
    assert "SANITIZED-OK" in r.stdout, report
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, report

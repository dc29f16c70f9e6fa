"""Pins for the oracle functions of SURVEY.md §8(f) NEXT-1..3: the paper's own indicator (averaged
finite-time velocity, central projection on S, density on the sphere), the drift detector
dP(t), the survivor filter and the uniform-on-sphere initial conditions.

As in test_oracle_pins.py nothing here compares the oracle with itself or with the CUDA path: closed
forms (eps = 0), a library routine on a special case (pendulum rotation frequency via ellipk), brute
force (an unwrapped run without checkpoints; a test-side re-binning; a stepwise survivor loop),
hand-made cases and statistics of the sampler.  Pin numbers P15.. continue DESIGN.md §4.
"""
import math

import numpy as np
import pytest

TWO_PI = 2.0 * math.pi


def _one(orc, q0, E, eps, order=4, wind=True):
    """A one-trajectory oracle State holding q0 (status live, H0 from the oracle's own routine)."""
    st = orc.State(1, tangent=False, wind=wind)
    st.q[:, 0] = q0
    st.status[0] = 1
    st.E, st.eps, st.order = E, eps, order
    st.acc[2, 0] = orc.hamiltonian(q0, eps)
    return st


# ------------------------------------------------------------------ P15: eps = 0, V = P exactly

@pytest.mark.parametrize("order", [4, 6])
def test_P15_free_motion_velocity_is_the_momentum(orc, order):
    """eps = 0: X(t) = X(0) + P t, so V = [X(t+Dt) - X(t)]/Dt = P, and since P^2 = 2E the central
    projection leaves it where it is.  400 checkpoints, ~130 whole turns: a dropped or mis-signed turn
    count, or a wrong Dt, fails this."""
    E = 1.0
    rng = np.random.default_rng(5)
    n = 64
    st = orc.State(n, tangent=False, wind=True)
    d = rng.normal(size=(3, n))
    d /= np.linalg.norm(d, axis=0)
    st.q[:3, :n] = rng.uniform(0, TWO_PI, (3, n))
    st.q[3:, :n] = math.sqrt(2 * E) * d
    st.status[:] = 1
    st.E, st.eps, st.order = E, 0.0, order
    orc.integrate(st, 300, 0.01, 100)            # the window does not start at t = 0
    orc.mark(st)
    orc.integrate(st, 40000, 0.01, 100)          # Dt = 400, |X| moves ~ 565 rad = 90 turns
    assert abs((st.t - st.tref) - 400.0) < 1e-9
    assert np.max(np.abs(st.wind[:, :n])) > 50
    V = orc.velocity(st, projected=False)
    Vh = orc.velocity(st, projected=True)
    assert np.max(np.abs(V - st.q[3:, :n])) < 1e-12
    assert np.max(np.abs(Vh - st.q[3:, :n])) < 1e-12
    # dP(t) = |P(t) - P(0)| = 0 exactly (P:37 with eps = 0)
    assert np.all(orc.delta_p(st) == 0.0)


# ------------------------------------------------------------------ P16: vs an unwrapped brute-force run

@pytest.mark.parametrize("order,eps", [(4, 3e-2), (6, 1e-2)])
def test_P16_velocity_equals_unwrapped_displacement(orc, order, eps):
    """eps > 0: the same trajectory integrated by oracle.steps (no checkpoint, no wrap, angles grow
    freely) gives X(t+Dt) - X(t) directly; the checkpointed run must reconstruct it from wrapped angles
    + turn counters.  Regular orbit, 2000 steps: the two runs differ by rounding only."""
    rng = np.random.default_rng(11)
    E, dt = 1.0, 0.01
    X = rng.uniform(0, TWO_PI, 3)
    pxy = np.array([0.37, -0.81])
    hp = math.cos(X[0]) * math.cos(X[1]) * (1 + math.cos(2 * X[2]))
    pz = math.sqrt(2 * (E - eps * hp) - pxy @ pxy)
    q0 = np.concatenate([X, pxy, [pz]])
    st = _one(orc, q0, E, eps, order)
    orc.mark(st)
    orc.integrate(st, 2000, dt, 100)
    qb, _ = orc.steps(q0, None, order, dt, eps, 2000)
    Vb = (qb[:3] - q0[:3]) / (2000 * dt)
    V = orc.velocity(st, projected=False)[:, 0]
    assert np.max(np.abs(V - Vb)) < 1e-11
    Vh = orc.velocity(st, projected=True)[:, 0]
    assert np.max(np.abs(Vh - math.sqrt(2 * E) * Vb / np.linalg.norm(Vb))) < 1e-11
    dp = orc.delta_p(st)[0]
    assert abs(dp - np.linalg.norm(qb[3:] - q0[3:])) < 1e-11 and dp > 1e-4


# ------------------------------------------------------------------ P17: pendulum rotation frequency

def test_P17_averaged_velocity_of_the_pendulum_is_2pi_over_T(orc):
    """On y = z = p_y = p_z = 0 the model is the pendulum H = p_x^2/2 + 2 eps cos x (P8).  Over exactly
    m rotation periods T(h) = 4 K(k^2)/sqrt(2 (h + 2 eps)) the angle advances by 2 pi m, so the averaged
    velocity is V_x = 2 pi / T(h) — a library routine (scipy.special.ellipk), not the integrator."""
    from scipy.special import ellipk
    eps, px0, E = 1e-2, 1.0, 0.52
    h = 0.5 * px0 ** 2 + 2 * eps
    T = 4 * ellipk(4 * eps / (h + 2 * eps)) / math.sqrt(2 * (h + 2 * eps))
    nper, nstep = 7, 7000
    st = _one(orc, np.array([0.0, 0, 0, px0, 0, 0]), E, eps, 6)
    orc.mark(st)
    orc.integrate(st, nstep, nper * T / nstep, 100)
    V = orc.velocity(st, projected=False)[:, 0]
    assert abs(V[0] - TWO_PI / T) < 1e-10
    assert V[1] == 0.0 and V[2] == 0.0
    # x = 0 is the top of the potential: p_x0 is the slowest speed, sqrt(2 (h + 2 eps)) the fastest
    assert px0 < V[0] < math.sqrt(2 * (h + 2 * eps))
    Vh = orc.velocity(st, projected=True)[:, 0]
    assert abs(Vh[0] - math.sqrt(2 * E)) < 1e-15 and Vh[1] == 0.0 and Vh[2] == 0.0


# ------------------------------------------------------------------ P18: central projection, hand case

def test_P18_central_projection_hand_case(orc):
    """fn. 26: Vhat = sqrt(2E) V/|V|.  Displacement (3, 4, 12) c over Dt has |V| = 13 c/Dt."""
    E, Dt = 8.0, 2.0                               # sqrt(2E) = 4
    st = _one(orc, np.array([0.1, 0.2, 0.3, 1, 1, 1.0]), E, 0.0)
    orc.mark(st)
    c = 0.01
    st.q[:3, 0] += c * np.array([3.0, 4.0, 12.0])
    st.wind[:, 0] += np.array([0, 0, 0])
    st.t = st.tref + Dt
    Vh = orc.velocity(st, projected=True)[:, 0]
    assert np.max(np.abs(Vh - 4.0 * np.array([3.0, 4.0, 12.0]) / 13.0)) < 1e-13
    # whole turns enter through the counters: one extra turn in y, wrapped angle unchanged
    st.wind[1, 0] += 1
    V = orc.velocity(st, projected=False)[:, 0]
    assert abs(V[1] - (0.04 + TWO_PI) / Dt) < 1e-14 and abs(V[0] - 0.03 / Dt) < 1e-15
    # |Vhat|^2 = 2E for anything
    Vh = orc.velocity(st, projected=True)[:, 0]
    assert abs(Vh @ Vh - 2 * E) < 1e-13
    # zero displacement: nothing to project -> NaN, and the density drops it
    st.q[:3, 0] = st.qref[:3, 0]
    st.wind[:, 0] = st.windref[:, 0]
    assert np.all(np.isnan(orc.velocity(st, projected=True)))
    hist = np.zeros((8, 8), dtype=np.uint32)
    d = orc.density_velocity(st, hist, -4.0, 4.0, hemi=3)
    assert hist.sum() == 0 and d[0] == 1


# ------------------------------------------------------------------ P19: density on the sphere, brute force

def test_P19_velocity_density_bruteforce_and_hemispheres(orc):
    """The histogram of (Vhat_x, Vhat_y) equals a test-side re-binning of the projected velocities
    (numpy floor on the same two roundings); hemispheres 1 + 2 = 3; sum + dropped = live count."""
    E, eps, G = 1.0, 2e-2, 64
    n = 48 * 40
    st = orc.State(n, tangent=False, wind=True)
    g = orc.make_grid(48, 40, -1.0, 1.0, angle_mode=1)
    orc.init_shell(st, g, E, eps, 3)
    st.q[5, : n // 2] *= -1.0                      # half of the ensemble on the lower hemisphere
    live = st.status == 1
    orc.mark(st)
    orc.integrate(st, 500, 0.01, 100)
    Vh = orc.velocity(st, projected=True)
    lo, hi = -1.5, 1.5
    hists, drops = {}, {}
    for hemi in (1, 2, 3):
        hists[hemi] = np.zeros((G, G), dtype=np.uint32)
        drops[hemi] = int(orc.density_velocity(st, hists[hemi], lo, hi, hemi)[0])
        assert int(hists[hemi].sum()) + drops[hemi] == int(live.sum())
    assert np.array_equal(hists[1] + hists[2], hists[3])
    assert hists[1].sum() > 0 and hists[2].sum() > 0
    f = G / (hi - lo)
    ix = np.floor((Vh[0] - lo) * f)
    iy = np.floor((Vh[1] - lo) * f)
    ok = live & np.isfinite(ix) & (ix >= 0) & (ix < G) & (iy >= 0) & (iy < G)
    for hemi, sel in ((1, Vh[2] >= 0), (2, Vh[2] < 0), (3, np.ones(n, bool))):
        ref = np.zeros((G, G), dtype=np.uint32)
        np.add.at(ref, (iy[ok & sel].astype(int), ix[ok & sel].astype(int)), 1)
        assert np.array_equal(ref, hists[hemi])
    # accumulates over calls (time-averaged density)
    again = hists[3].copy()
    orc.density_velocity(st, again, lo, hi, 3)
    assert np.array_equal(again, 2 * hists[3])
    # regular orbits stay "at the close vicinity of the initial momentum vector": for most of the
    # ensemble the projected averaged velocity is within a few eps of the projected initial momentum
    P0 = st.qref[3:, :n]
    P0h = math.sqrt(2 * E) * P0 / np.linalg.norm(P0, axis=0)
    dist = np.linalg.norm(Vh - P0h, axis=0)[live]
    assert np.median(dist) < 5 * eps


# ------------------------------------------------------------------ P20: sticking to a resonance

def test_P20_resonant_orbit_velocity_obeys_the_resonance_condition(orc):
    """inside the layer of resonance m the system moves with m . V ~ 0.  An orbit started inside the
    island of Omega_(1,-1,0) (p_x - p_y = 0.01, well below the island half-width ~ 2 sqrt(2 eps) = 0.28,
    at the stable phase x - y = pi of the resonant term (eps/2) cos(x - y)(1 + cos 2z)) librates:
    averaged over 200 time units |V_x - V_y| is far below |p_x - p_y|(0); an orbit outside the island
    (p_x - p_y = 0.6) keeps V_x - V_y close to its initial value."""
    E, eps = 1.0, 1e-2

    def run(dp):
        px, py = 0.5 + dp / 2, 0.5 - dp / 2
        X = np.array([math.pi, 0.0, 0.4])
        hp = math.cos(X[0]) * math.cos(X[1]) * (1 + math.cos(2 * X[2]))
        pz = math.sqrt(2 * (E - eps * hp) - px * px - py * py)
        st = _one(orc, np.concatenate([X, [px, py, pz]]), E, eps, 4)
        orc.mark(st)
        orc.integrate(st, 20000, 0.01, 100)
        return orc.velocity(st, projected=False)[:, 0]

    Vin = run(0.01)
    assert abs(Vin[0] - Vin[1]) < 2e-3
    Vout = run(0.6)
    assert abs((Vout[0] - Vout[1]) - 0.6) < 0.05


# ------------------------------------------------------------------ P21: survivor filter

def test_P21_survivor_filter_vs_stepwise_bruteforce(orc):
    """A trajectory is dropped (status 3, frozen) at the first checkpoint at which (p_x, p_y) is outside
    the launch rectangle.  Brute force: the same ensemble without the filter, advanced one stride at a
    time, with the test deciding when each trajectory left."""
    E, eps, n = 1.0, 3e-2, 32 * 32
    rect = (-0.2, 0.2, -0.2, 0.2)
    g = orc.make_grid(32, 32, rect[0], rect[1], angle_mode=1)
    a = orc.State(n, tangent=False, wind=True)
    orc.init_shell(a, g, E, eps, 9)
    b = a.copy()
    a.surv = rect
    orc.integrate(a, 3000, 0.01, 100)
    left_at = np.full(n, -1)
    frozen = np.zeros((6, n))
    for c in range(30):
        orc.integrate(b, 100, 0.01, 100)
        px, py = b.q[3, :n], b.q[4, :n]
        out = ~((px >= rect[0]) & (px < rect[1]) & (py >= rect[2]) & (py < rect[3]))
        new = out & (left_at < 0)
        left_at[new] = c
        frozen[:, new] = b.q[:, :n][:, new]
    gone = left_at >= 0
    assert 0 < gone.sum() < n                                  # the case is not degenerate
    assert np.array_equal(a.status == 3, gone)
    assert np.array_equal(a.status == 1, ~gone)
    assert np.array_equal(a.q[:, :n][:, gone], frozen[:, gone])        # frozen where it left
    assert np.array_equal(a.q[:, :n][:, ~gone], b.q[:, :n][:, ~gone])  # survivors untouched by the filter
    # dropped trajectories are not counted by the densities or the images
    hist = np.zeros((16, 16), dtype=np.uint32)
    d = orc.density(a, hist, -1.0, 1.0)
    assert int(hist.sum()) + int(d[0]) == int((~gone).sum())
    # eps = 0: P is constant, nobody ever leaves
    c0 = orc.State(n, tangent=False, wind=True)
    orc.init_shell(c0, g, E, 0.0, 9)
    c0.surv = rect
    orc.integrate(c0, 1000, 0.01, 100)
    assert np.all(c0.status == 1)
    # single checkpoint, hand-made: on the upper edge (half-open) -> dropped; just inside -> kept
    q = np.array([0.1, 0.2, 0.3, 0.2, 0.0, 1.0])
    assert orc.checkpoint(q, None, np.zeros(4), None, 0.0, rect)[4] == 3
    q[3] = np.nextafter(0.2, 0.0)
    assert orc.checkpoint(q, None, np.zeros(4), None, 0.0, rect)[4] == 1
    q[3] = -0.2
    assert orc.checkpoint(q, None, np.zeros(4), None, 0.0, rect)[4] == 1


# ------------------------------------------------------------------ P22: uniform on the sphere S

def test_P22_sphere_initial_conditions(orc):
    """"initial conditions uniformly distributed over the sphere S, and over the torus".  Every
    point is on the shell (|H0 - E| <= 16 ulp: three rounded squares and their sums; never masked); the direction is uniform: cos(theta) is
    uniform on [-1, 1] (chi-square over 32 equal-area bands), phi uniform, <p_i p_j>/2E = delta_ij/3."""
    for E, eps in ((400.0, 1.0), (15.0, 1.0), (1.0, 3e-2)):
        n = 1 << 16
        st = orc.State(n, tangent=False, wind=True)
        g = orc.make_grid(256, 256, angle_mode=1, shape=3)
        orc.init_shell(st, g, E, eps, 12345)
        assert np.all(st.status == 1)
        assert np.max(np.abs(st.acc[2, :n] - E)) <= 16 * np.spacing(E)
        P = st.q[3:, :n]
        X = st.q[:3, :n]
        hp = np.cos(X[0]) * np.cos(X[1]) * (1 + np.cos(2 * X[2]))
        assert np.max(np.abs(np.sum(P * P, axis=0) - 2 * (E - eps * hp))) < 1e-12 * E
        d = P / np.linalg.norm(P, axis=0)
        cnt, _ = np.histogram(d[2], bins=32, range=(-1, 1))
        chi2 = np.sum((cnt - n / 32) ** 2 / (n / 32))
        assert chi2 < 70.0                                      # 31 dof: P(chi2 > 70) ~ 1e-4
        phi = np.arctan2(d[1], d[0])
        cnt, _ = np.histogram(phi, bins=32, range=(-math.pi, math.pi))
        assert np.sum((cnt - n / 32) ** 2 / (n / 32)) < 70.0
        C = d @ d.T / n
        assert np.max(np.abs(C - np.eye(3) / 3)) < 4.0 / math.sqrt(n)
        # both hemispheres are populated; pz_sign = -1 mirrors the third action only
        assert 0.45 < np.mean(P[2] > 0) < 0.55
    st2 = orc.State(n, tangent=False, wind=True)
    orc.init_shell(st2, orc.make_grid(256, 256, angle_mode=1, shape=3, pz_sign=-1), 1.0, 3e-2, 12345)
    assert np.array_equal(st2.q[5, :n], -st.q[5, :n]) and np.array_equal(st2.q[:5, :n], st.q[:5, :n])


# ------------------------------------------------------------------ P23: energy-drift statistics (configs[2])

def test_P23_energy_drift_statistics(orc):
    """max / mean / rms of dH_max and mean / rms of the signed final error H(t) - H0 over the live trajectories:
    (i) against numpy on the images (test-side arithmetic, mpmath H on a few pixels); (ii) eps = 0: every entry
    is at the rounding level; (iii) P:55 "no secular growth": doubling the horizon leaves max dH_max within a
    factor 1.5 and the signed mean stays far below the rms; (iv) order 6 beats order 4 by > 100 at dt = 0.02."""
    import mpmath as mp
    mp.mp.dps = 30
    E, eps = 1.0, 1e-2
    n = 40 * 30
    st = orc.State(n, tangent=False, wind=True)
    orc.init_shell(st, orc.make_grid(40, 30, -1.04, 1.04, angle_mode=1), E, eps, 21)
    orc.integrate(st, 2000, 0.02, 100)
    out, img = orc.energy_stats(st)
    live = st.status == 1
    assert 0 < (~live).sum() < n and np.all(np.isnan(img[~live])) and not np.any(np.isnan(img[live]))
    d = st.acc[3, :n][live]
    assert out[0] == live.sum() and out[1] == d.max()
    assert abs(out[2] - d.mean()) < 1e-12 * d.mean() and abs(out[3] - math.sqrt((d * d).mean())) < 1e-12 * out[3]
    assert np.nonzero(live)[0][np.argmax(d)] == int(out[6])
    sd = img[live]
    assert abs(out[4] - sd.mean()) < 1e-18 + 1e-9 * abs(sd).max() and abs(out[5] - math.sqrt((sd * sd).mean())) < 1e-12 * out[5]
    assert out[7] == np.abs(sd).max() and out[7] <= out[1] * (1 + 1e-9) + 1e-15   # the final state is one sample
    for k in np.nonzero(live)[0][:20]:
        x, y, z, px, py, pz = (mp.mpf(float(v)) for v in st.q[:, k])
        H = (px * px + py * py + pz * pz) / 2 + mp.mpf(eps) * mp.cos(x) * mp.cos(y) * (1 + mp.cos(2 * z))
        assert abs(float(H - mp.mpf(float(st.acc[2, k]))) - img[k]) < 4e-16
    # (iii) no secular growth
    max1, mean_signed1 = out[1], out[4]
    orc.integrate(st, 2000, 0.02, 100)
    out2, _ = orc.energy_stats(st)
    assert out2[1] < 1.5 * max1
    assert abs(out2[4]) < 0.5 * out2[5]
    # (iv) order
    s6 = orc.State(n, tangent=False, wind=True)
    orc.init_shell(s6, orc.make_grid(40, 30, -1.04, 1.04, angle_mode=1), E, eps, 21)
    s6.order = 6
    orc.integrate(s6, 2000, 0.02, 100)
    assert orc.energy_stats(s6)[0][1] < max1 / 100
    # (ii) eps = 0
    s0 = orc.State(n, tangent=False, wind=True)
    orc.init_shell(s0, orc.make_grid(40, 30, -0.9, 0.9, angle_mode=1), E, 0.0, 21)
    orc.integrate(s0, 1000, 0.02, 100)
    o0, i0 = orc.energy_stats(s0)
    assert o0[0] == n and o0[1] == 0.0 and o0[7] == 0.0 and np.all(i0 == 0.0)
    # empty ensemble: count 0, NaN means
    e = orc.State(4, tangent=False, wind=True)
    oe, _ = orc.energy_stats(e)
    assert oe[0] == 0 and np.isnan(oe[2]) and oe[6] == -1

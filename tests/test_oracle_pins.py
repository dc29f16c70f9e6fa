"""Pins for the parity oracle (oracle/aw_oracle.cpp) against what the paper and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path: each is a closed form, an
invariant, a library routine on a special case, a finite-difference brute force, or a value the paper
prints (tests/golden/paper_values.txt).  Pin numbers P1..P13 follow DESIGN.md §5.
PAPER.md citations: P:<line>.
"""
import math
import os

import numpy as np
import pytest

TWO_PI = 2.0 * math.pi
RNG = np.random.default_rng(20110721)


def golden():
    out = {}
    path = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")
    for line in open(path):
        line = line.split("#")[0].split()
        if line:
            out[line[0]] = [float(v) for v in line[1:]]
    return out


def shell_state(E, eps, orc, rng=RNG):
    """A random state with H = E: random angles and direction, |P| from eq. (1) (test-side arithmetic)."""
    X = rng.uniform(0, TWO_PI, 3)
    d = rng.normal(size=3)
    d /= np.linalg.norm(d)
    hp = math.cos(X[0]) * math.cos(X[1]) * (1 + math.cos(2 * X[2]))
    return np.concatenate([X, math.sqrt(2 * (E - eps * hp)) * d])


# ------------------------------------------------------------------ model: eq. (1), (2)

def test_model_values_and_bounds(orc):
    g = golden()
    # eq. (2) at hand-computable points
    assert orc.hp(0.0, 0.0, 0.0) == 2.0                      # maximum, |H_p| <= 2
    assert abs(orc.hp(math.pi, 0.0, 0.0) + 2.0) < 1e-15      # minimum at (pi, 0, 0)
    assert abs(orc.hp(0.3, 0.0, math.pi / 2)) < 1e-15        # 1 + cos(pi) = 0
    assert abs(orc.hp(math.pi / 3, math.pi / 3, math.pi / 6) - 0.25 * 1.5) < 1e-15
    pts = RNG.uniform(-10, 10, (2000, 3))
    vals = np.array([orc.hp(*p) for p in pts])
    assert np.all(np.abs(vals) <= g["hp_bound"][0])
    # retyped eq. (2) with mpmath at 30 digits (independent arithmetic)
    import mpmath as mp
    mp.mp.dps = 30
    for p in pts[:50]:
        ref = mp.cos(mp.mpf(p[0])) * mp.cos(mp.mpf(p[1])) * (1 + mp.cos(2 * mp.mpf(p[2])))
        assert abs(orc.hp(*p) - float(ref)) < 4e-16
    # eq. (1): kinetic part
    q = np.array([0.3, 0.0, math.pi / 2, 1.0, 2.0, -2.0])
    assert abs(orc.hamiltonian(q, 0.7) - 4.5) < 1e-15
    # eq. (3): eps_eff = 2/E values the paper prints
    assert g["eps_eff_E400"][0] == 2.0 / 400.0
    assert g["eps_eff_E15"][0] == 2.0 / 15.0


def test_gradient_and_hessian_vs_central_differences(orc):
    h = 1e-5
    for p in RNG.uniform(-4, 4, (40, 3)):
        g = orc.grad(*p)
        H = orc.hess(*p)
        assert np.array_equal(H, H.T)
        for i in range(3):
            e = np.zeros(3)
            e[i] = h
            fd = (orc.hp(*(p + e)) - orc.hp(*(p - e))) / (2 * h)
            assert abs(g[i] - fd) < 2e-9
            fdg = (orc.grad(*(p + e)) - orc.grad(*(p - e))) / (2 * h)
            assert np.max(np.abs(H[i] - fdg)) < 2e-9


# ------------------------------------------------------------------ P4 coefficients

def test_P4_order_conditions(orc):
    import mpmath as mp
    mp.mp.dps = 40
    for order, S in ((4, 3), (6, 7), (66, 9)):
        w = [mp.mpf(float(v)) for v in orc.stage_list(order)]
        assert len(w) == S
        assert w == w[::-1]                                   # palindromic => symmetric => even order
        assert abs(sum(w) - 1) < 1e-15
        assert abs(sum(x ** 3 for x in w)) < 2e-14   # rounding of w to double: 3 w^2 ulp(w)
        if order >= 6:
            assert abs(sum(x ** 5 for x in w)) < 2e-13   # 5 w^4 ulp(w), |w| up to 3 for the 9-stage list
            acc, pre = mp.mpf(0), mp.mpf(0)
            for x in w:
                acc += x ** 3 * (pre + x / 2) ** 2
                pre += x
            assert abs(acc) < 2e-13
    # closed forms for the triple jump (order 4)
    w4 = orc.stage_list(4)
    assert abs(w4[0] - 1 / (2 - 2 ** (1 / 3))) < 1e-15 and abs(w4[1] + 2 ** (1 / 3) / (2 - 2 ** (1 / 3))) < 1e-15
    # drift constants sum to dt, kick constants to eps*dt
    for order in (4, 6):
        a, b = orc.stage_constants(order, 0.01, 0.03)
        assert abs(a.sum() - 0.01) < 1e-17 and abs(b.sum() - 0.03 * 0.01) < 1e-18
        assert len(a) == len(b) + 1


# ------------------------------------------------------------------ P1, P2: eps = 0

@pytest.mark.parametrize("order", [4, 6])
def test_P1_free_motion_closed_form(orc, order):
    q0 = np.array([0.1, -2.0, 3.0, 0.7, -1.1, 0.4])
    n, dt = 1000, 0.01
    q, _ = orc.steps(q0, None, order, dt, 0.0, n)
    assert np.array_equal(q[3:], q0[3:])                      # P bit-constant
    exact = q0[:3] + n * dt * q0[3:]                          # X(t) = X(0) + P t
    assert np.max(np.abs(q[:3] - exact)) < n * 8 * np.finfo(float).eps * 4


@pytest.mark.parametrize("order", [4, 6])
def test_P2_free_tangent_and_fli_closed_form(orc, order):
    n, dt, stride = 2000, 0.01, 100
    st = orc.State(1, tangent=True, wind=True)
    q0 = np.array([0.1, -2.0, 3.0, 0.7, -1.1, 0.4])
    w0 = np.array([0.3, -0.2, 0.1, 0.5, 0.4, -0.66])
    w0 /= np.linalg.norm(w0)
    st.q[:, 0], st.w[:, 0], st.status[0] = q0, w0, 1
    st.eps, st.order = 0.0, order
    st.acc[2, 0] = orc.hamiltonian(q0, 0.0)
    orc.integrate(st, n, dt, stride)
    t = n * dt
    # closed form: dP const, dX(t) = dX0 + t dP0; logsum(t) = ln |w(t)| because renormalisation is linear
    norms = [math.sqrt(np.sum((w0[:3] + tt * w0[3:]) ** 2) + np.sum(w0[3:] ** 2))
             for tt in np.arange(1, n // stride + 1) * stride * dt]
    assert abs(st.acc[0, 0] - math.log(norms[-1])) < 1e-12
    assert abs(st.acc[1, 0] - max(0.0, max(math.log(v) for v in norms))) < 1e-12
    wt = np.concatenate([w0[:3] + t * w0[3:], w0[3:]])
    assert np.max(np.abs(st.w[:, 0] - wt / np.linalg.norm(wt))) < 1e-13
    assert abs(np.linalg.norm(st.w[:, 0]) - 1) < 1e-15
    # angles: wrapped value + 2 pi wind equals the free-motion closed form
    X = st.q[:3, 0] + TWO_PI * st.wind[:, 0]
    assert np.max(np.abs(X - (q0[:3] + t * q0[3:]))) < 1e-12
    assert np.all(np.abs(st.q[:3, 0]) <= math.pi + 1e-15)
    assert st.acc[3, 0] == 0.0                                # H = P^2/2 is exactly conserved
    assert orc.indicator(st, 1)[0] == st.acc[0, 0] / t        # FTLE = logsum / t


# ------------------------------------------------------------------ P3: order of the scheme

def max_dh(orc, order, dt, T, q0, eps):
    n = int(round(T / dt))
    h0 = orc.hamiltonian(q0, eps)
    q, worst = q0.copy(), 0.0
    for _ in range(20):
        q, _ = orc.steps(q, None, order, dt, eps, n // 20)
        worst = max(worst, abs(orc.hamiltonian(q, eps) - h0))
    return worst


@pytest.mark.parametrize("order,expect,tol", [(2, 4.0, 0.6), (4, 16.0, 3.0), (6, 64.0, 14.0), (66, 64.0, 14.0)])
def test_P3_energy_error_order(orc, order, expect, tol):
    eps, E = 1e-2, 1.0
    rng = np.random.default_rng(3)
    ics = [shell_state(E, eps, orc, rng) for _ in range(24)]
    dts = [0.4, 0.2, 0.1]
    errs = [max(max_dh(orc, order, dt, 40.0, q0, eps) for q0 in ics) for dt in dts]
    ratios = [errs[i] / errs[i + 1] for i in range(len(dts) - 1)]
    for r in ratios:
        assert abs(r - expect) < tol, (order, errs, ratios)


def test_P3b_sixth_order_schemes_agree(orc):
    """Yoshida solution A (7 stages) and the closed-form 9-stage triple jump are both 6th order:
    after one step they differ by O(dt^7), i.e. x128 per doubling of dt."""
    eps = 0.05
    q0 = shell_state(1.0, eps, orc, np.random.default_rng(5))
    d = []
    for dt in (0.2, 0.4):
        qa, _ = orc.steps(q0, None, 6, dt, eps, 1)
        qb, _ = orc.steps(q0, None, 66, dt, eps, 1)
        d.append(np.max(np.abs(qa - qb)))
    assert 90 < d[1] / d[0] < 180, d


# ------------------------------------------------------------------ P5: reversibility

@pytest.mark.parametrize("order", [4, 6])
def test_P5_time_reversibility(orc, order):
    eps = 1e-2
    rng = np.random.default_rng(7)
    for _ in range(8):
        q0 = shell_state(1.0, eps, orc, rng)
        q, _ = orc.steps(q0, None, order, 0.01, eps, 1000)
        assert np.max(np.abs(q - q0)) > 1e-3
        q, _ = orc.steps(q, None, order, -0.01, eps, 1000)
        assert np.max(np.abs(q - q0)) < 1e-12
    # through the checkpointed path (wraps + winding counters): compare X + 2 pi wind
    st = orc.State(4, tangent=False, wind=True)
    for k in range(4):
        st.q[:, k] = shell_state(1.0, eps, orc, rng)
        st.status[k] = 1
        st.acc[2, k] = orc.hamiltonian(st.q[:, k], eps)
    st.eps, st.order = eps, order
    q0 = st.q.copy()
    orc.integrate(st, 1000, 0.01, 100)
    orc.integrate(st, 1000, -0.01, 100)
    X = st.q[:3, :4] + TWO_PI * st.wind[:, :4]
    assert np.max(np.abs(X - q0[:3, :4])) < 1e-12
    assert np.max(np.abs(st.q[3:, :4] - q0[3:, :4])) < 1e-12


# ------------------------------------------------------------------ P6, P7: tangent map

@pytest.mark.parametrize("order", [4, 6])
def test_P6_tangent_map_is_symplectic(orc, order):
    eps = 3e-2
    q0 = shell_state(1.0, eps, orc, np.random.default_rng(11))
    M = np.zeros((6, 6))
    for j in range(6):
        e = np.zeros(6)
        e[j] = 1.0
        _, w = orc.steps(q0, e, order, 0.01, eps, 1000)
        M[:, j] = w
    J = np.zeros((6, 6))
    J[:3, 3:] = np.eye(3)
    J[3:, :3] = -np.eye(3)
    assert np.max(np.abs(M.T @ J @ M - J)) < 1e-12
    assert abs(np.linalg.det(M) - 1.0) < 1e-12
    assert np.max(np.abs(M - np.eye(6))) > 0.1                # not trivially the identity


@pytest.mark.parametrize("order", [4, 6])
def test_P7_tangent_is_derivative_of_the_map(orc, order):
    eps, delta = 3e-2, 1e-7
    rng = np.random.default_rng(13)
    q0 = shell_state(1.0, eps, orc, rng)
    w0 = rng.normal(size=6)
    w0 /= np.linalg.norm(w0)
    qa, w = orc.steps(q0, w0, order, 0.01, eps, 500)
    qp, _ = orc.steps(q0 + delta * w0, None, order, 0.01, eps, 500)
    qm, _ = orc.steps(q0 - delta * w0, None, order, 0.01, eps, 500)
    fd = (qp - qm) / (2 * delta)
    assert np.max(np.abs(fd - w)) / np.max(np.abs(w)) < 1e-6


# ------------------------------------------------------------------ P8: pendulum reduction vs ellipk

@pytest.mark.parametrize("order,rtol", [(4, 2e-9), (6, 1e-11)])
def test_P8_pendulum_period_vs_elliptic_integral(orc, order, rtol):
    """y = z = p_y = p_z = 0 is invariant; there H = p_x^2/2 + 2 eps cos x (a pendulum).  For a rotating
    orbit of energy h the period of x -> x + 2 pi is T = 4 K(m) / sqrt(2 (h + 2 eps)), m = 4 eps/(h + 2 eps)
    (scipy.special.ellipk takes the parameter m = k^2)."""
    from scipy.special import ellipk
    eps, px0 = 1e-2, 1.0
    h = 0.5 * px0 ** 2 + 2 * eps
    m = 4 * eps / (h + 2 * eps)
    T = 4 * ellipk(m) / math.sqrt(2 * (h + 2 * eps))
    n = 2000
    q0 = np.array([0.0, 0.0, 0.0, px0, 0.0, 0.0])
    q, _ = orc.steps(q0, None, order, T / n, eps, n)
    assert abs(q[0] - TWO_PI) < rtol * TWO_PI
    assert abs(q[3] - px0) < rtol
    assert np.all(q[[1, 2, 4, 5]] == 0.0)                     # invariant subspace, exactly


# ------------------------------------------------------------------ P9: invariant subspaces, symmetries

@pytest.mark.parametrize("order", [4, 6])
def test_P9_invariant_subspaces_and_symmetries(orc, order):
    eps = 3e-2
    q0 = np.array([0.4, -1.3, 0.0, 0.9, 0.5, 0.0])            # 2-D limit z = 0, p_z = 0
    q, _ = orc.steps(q0, None, order, 0.01, eps, 3000)
    assert q[2] == 0.0 and q[5] == 0.0
    assert abs(q[0] - q0[0] - 30 * q0[3]) < 1.0               # moved, roughly ballistically
    r = shell_state(1.0, eps, orc, np.random.default_rng(17))
    qa, _ = orc.steps(r, None, order, 0.01, eps, 500)
    qb, _ = orc.steps(r[[1, 0, 2, 4, 3, 5]], None, order, 0.01, eps, 500)   # x <-> y swap
    assert np.max(np.abs(qb[[1, 0, 2, 4, 3, 5]] - qa)) < 1e-12
    qc, _ = orc.steps(-r, None, order, 0.01, eps, 500)                       # X,P -> -X,-P
    assert np.array_equal(qc, -qa)


# ------------------------------------------------------------------ scaling equivalence (eq. 3, D2)

def test_energy_vs_eps_parametrisations_are_the_same_family(orc):
    """(E, eps = 1), the paper's choice, equals (E' = 1, eps' = 1/E) after P = sqrt(E) P',
    t = t'/sqrt(E): same X at every step, momenta scaled by sqrt(E)."""
    E = 15.0
    rng = np.random.default_rng(19)
    q0 = shell_state(E, 1.0, orc, rng)
    q1 = q0.copy()
    q1[3:] /= math.sqrt(E)
    assert abs(orc.hamiltonian(q1, 1.0 / E) - 1.0) < 1e-14
    dt = 0.01
    qa, _ = orc.steps(q0, None, 6, dt / math.sqrt(E), 1.0, 400)
    qb, _ = orc.steps(q1, None, 6, dt, 1.0 / E, 400)
    assert np.max(np.abs(qa[:3] - qb[:3])) < 1e-11
    assert np.max(np.abs(qa[3:] / math.sqrt(E) - qb[3:])) < 1e-12


# ------------------------------------------------------------------ P10, P11: shell and ICs

def test_P11_init_shell_grid(orc):
    eps = 5e-2
    g = orc.make_grid(64, 64, angle_mode=1)
    st = orc.init_shell(orc.State(64 * 64), g, 1.0, eps, 0)
    n = st.n
    live = st.status == 1
    assert live.sum() > 0.9 * n and (~live).sum() > 0        # corners of [-1,1]^2: some off shell (R8)
    # cell-centred samples = histogram bin centres; k = j*gx + i, i <-> p_x fast (R6)
    k = 5 * 64 + 9
    assert st.q[3, k] == -1.0 + 9.5 * 2.0 / 64 and st.q[4, k] == -1.0 + 5.5 * 2.0 / 64
    # energy: recomputed here from eq. (1),(2) in plain numpy
    X, P = st.q[:3, :n], st.q[3:, :n]
    H = 0.5 * (P ** 2).sum(0) + eps * np.cos(X[0]) * np.cos(X[1]) * (1 + np.cos(2 * X[2]))
    assert np.max(np.abs(H[live] - 1.0)) <= 4 * np.finfo(float).eps
    assert np.max(np.abs(st.acc[2, :n][live] - 1.0)) <= 4 * np.finfo(float).eps
    assert np.all(P[2][live] >= 0)                            # + root (R9)
    # angles are 2pi_hi * u(seed, k, slot 0..2)
    u = np.array([[orc.uniform(0, kk, s) for s in range(3)] for kk in range(n)])
    ang = 6.283185307179586 * u
    assert np.array_equal(X.T[live], ang[live])
    # status 0 <=> negative radicand; those states are NaN
    px = -1.0 + (np.arange(n) % 64 + 0.5) * 2.0 / 64
    py = -1.0 + (np.arange(n) // 64 + 0.5) * 2.0 / 64
    R = 2 * (1.0 - eps * np.cos(ang[:, 0]) * np.cos(ang[:, 1]) * (1 + np.cos(2 * ang[:, 2]))) - px ** 2 - py ** 2
    clear = np.abs(R) > 1e-12
    assert np.array_equal((R >= 0)[clear], live[clear])
    assert np.all(np.isnan(st.q[:, :n][:, ~live])) and np.all(np.isnan(st.acc[2, :n][~live]))
    # angles 0 at eps = 1e-2 on this grid: p_x^2 + p_y^2 <= 2*0.984^2 = 1.94 < 2 - 4 eps: all on shell
    s0 = orc.init_shell(orc.State(n), orc.make_grid(64, 64), 1.0, 1e-2, 0)
    assert np.all(s0.status == 1) and np.all(s0.q[:3] == 0.0)
    # common tangent vector: unit norm, same for all
    assert abs(np.linalg.norm(st.w[:, 0]) - 1) < 1e-15
    assert np.array_equal(st.w[:, :n], np.repeat(st.w[:, :1], n, axis=1))
    assert np.array_equal(st.w[:, 0], orc.common_tangent(0))
    assert not np.array_equal(orc.common_tangent(0), orc.common_tangent(1))


def test_P11b_init_shell_cloud_and_modes(orc):
    n = 1 << 14
    g = orc.make_grid(128, 128, angle_mode=1, shape=1, cx=0.0, cy=0.0, r=1e-3, tangent_mode=1)
    st = orc.init_shell(orc.State(n), g, 1.0, 1e-3, 0)
    assert np.all(st.status == 1)
    rad = np.hypot(st.q[3, :n], st.q[4, :n])
    assert rad.max() <= 1e-3 and rad.max() > 0.99e-3
    # uniform in the disk: fraction inside r/2 is 1/4
    assert abs((rad < 0.5e-3).mean() - 0.25) < 0.02
    assert np.max(np.abs(np.linalg.norm(st.w[:, :n], axis=0) - 1)) < 1e-15
    assert np.abs(st.w[:, :n].mean(1)).max() < 0.02           # isotropic
    # p_z sign flag and Gaussian cloud
    g2 = orc.make_grid(128, 128, angle_mode=1, shape=2, cx=0.5, cy=-0.25, r=0.01, pz_sign=-1)
    s2 = orc.init_shell(orc.State(n), g2, 1.0, 1e-3, 3)
    assert np.all(s2.q[5, :n] < 0)
    assert abs(s2.q[3, :n].mean() - 0.5) < 5e-4 and abs(s2.q[4, :n].std() - 0.01) < 3e-4


def test_uniform_generator_statistics(orc):
    n = 1 << 16
    u = np.array([orc.uniform(42, k, 1) for k in range(n)])
    assert u.min() >= 0.0 and u.max() < 1.0
    counts = np.histogram(u, bins=64, range=(0, 1))[0]
    chi2 = ((counts - n / 64) ** 2 / (n / 64)).sum()
    assert chi2 < 120                                          # 63 dof: mean 63, sd 11
    v = np.array([orc.uniform(43, k, 1) for k in range(n)])
    assert abs(np.corrcoef(u, v)[0, 1]) < 0.02
    assert abs(np.corrcoef(u[:-1], u[1:])[0, 1]) < 0.02
    # u = (z >> 11) * 2^-53 of the 64-bit mixer
    assert orc.uniform(7, 5, 2) == (orc.mix64(7, 16 * 5 + 2) >> 11) * 2.0 ** -53


@pytest.mark.parametrize("order", [4, 6])
def test_P10_shell_layer_and_energy_bound(orc, order):
    """the dynamics stays in the layer 2(E - eps_eff) <= P^2 <= 2(E + eps_eff); in E = 1 units
    eps_eff*E = 2 eps.  Also: no secular energy growth."""
    eps = 3e-2
    g = orc.make_grid(16, 16, angle_mode=1)
    st = orc.init_shell(orc.State(256, tangent=False), g, 1.0, eps, 2)
    st.order = order
    worst = []
    for _ in range(5):
        orc.integrate(st, 2000, 0.01, 100)
        live = st.status == 1
        P2 = (st.q[3:, :256] ** 2).sum(0)[live]
        d = 2 * st.acc[3, :256][live]
        assert np.all(P2 >= 2 * (1.0 - 2 * eps) - d) and np.all(P2 <= 2 * (1.0 + 2 * eps) + d)
        worst.append(st.acc[3, :256][live].max())
    assert worst[-1] < (1e-9 if order == 4 else 1e-12)
    assert worst[-1] <= 3 * worst[0]                          # bounded, not growing with t


# ------------------------------------------------------------------ checkpoint: wrap and renormalisation

def test_checkpoint_wrap_and_renorm(orc):
    q = np.array([100.0, -7.0, 3.0, 0.1, 0.2, 0.3])
    w = np.array([3.0, 0.0, 4.0, 0.0, 0.0, 0.0])
    acc = np.array([0.5, 0.7, orc.hamiltonian(q, 0.1), 0.0])
    q2, w2, acc2, wind2, st = orc.checkpoint(q, w, acc, np.array([1, 2, 3], dtype=np.int32), 0.1)
    assert st == 1
    assert np.array_equal(wind2, [1 + 16, 2 - 1, 3 + 0])       # 100/2pi = 15.9 -> 16 ; -7/2pi = -1.1 -> -1
    import mpmath as mp
    mp.mp.dps = 40
    assert abs(q2[0] - float(mp.mpf(100) - 16 * 2 * mp.pi)) < 1e-15
    assert abs(q2[1] - float(mp.mpf(-7) + 2 * mp.pi)) < 1e-15
    assert q2[2] == 3.0 and np.array_equal(q2[3:], q[3:])
    assert np.allclose(w2, [0.6, 0, 0.8, 0, 0, 0], atol=1e-16)
    assert abs(acc2[0] - (0.5 + math.log(5.0))) < 1e-15 and acc2[1] == acc2[0]
    assert acc2[3] < 1e-15
    # non-finite state is flagged
    q[4] = float("inf")
    assert orc.checkpoint(q, None, acc, None, 0.1)[4] == 2


# ------------------------------------------------------------------ P12: histogram

def test_P12_density_bruteforce_and_edges(orc):
    n, G = 50000, 64
    st = orc.State(n, tangent=False)
    rng = np.random.default_rng(23)
    st.q[3, :n] = rng.uniform(-1.2, 1.2, n)
    st.q[4, :n] = rng.uniform(-1.2, 1.2, n)
    st.status[:] = 1
    st.status[::7] = 0
    hist = np.zeros((G, G), dtype=np.uint32)
    dropped = orc.density(st, hist, -1.0, 1.0)
    live = st.status == 1
    px, py = st.q[3, :n][live], st.q[4, :n][live]
    ref, _, _ = np.histogram2d(py, px, bins=G, range=[[-1, 1], [-1, 1]])
    # numpy's last bin is closed at +1; ours is half-open.  No sample sits exactly on +1 here.
    assert np.array_equal(hist, ref.astype(np.uint32))
    assert hist.sum() + dropped[0] == live.sum()
    # serial brute force
    brute = np.zeros((G, G), dtype=np.uint32)
    for x, y in zip(px, py):
        ix, iy = math.floor((x + 1) * G / 2), math.floor((y + 1) * G / 2)
        if 0 <= ix < G and 0 <= iy < G:
            brute[iy, ix] += 1
    assert np.array_equal(hist, brute)
    # accumulation across calls
    orc.density(st, hist, -1.0, 1.0, dropped)
    assert np.array_equal(hist, 2 * brute) and dropped[0] == 2 * (live.sum() - brute.sum())
    # hand-made edges on a 1024 grid: half-open bins [lo + i w, lo + (i+1) w)
    G = 1024
    # (p - lo) is rounded before the multiply (R20): 1 - 2^-52 -> 2 - 2^-52 exactly -> bin 1023, but
    # 1 - 2^-53 -> 2 - 2^-53 is a tie that rounds to 2.0 -> index 1024 -> dropped, like p = 1 itself.
    edge = np.array([-1.0, 1.0 - 2.0 ** -52, 1.0 - 2.0 ** -53, 1.0, -0.0, 2.0 / 1024, -2.0 / 1024,
                     np.nextafter(-1.0, -2.0)])
    st = orc.State(len(edge), tangent=False)
    st.q[3, :len(edge)] = edge
    st.q[4, :len(edge)] = 0.0
    st.status[:] = 1
    hist = np.zeros((G, G), dtype=np.uint32)
    dropped = orc.density(st, hist, -1.0, 1.0)
    row = hist[512]
    assert row[0] == 1 and row[1023] == 1 and row[512] == 1 and row[513] == 1 and row[511] == 1
    assert hist.sum() == 5 and dropped[0] == 3


# ------------------------------------------------------------------ P13: FLI ridge

def test_P13_fli_ridge_on_the_primary_resonance(orc):
    """Angles 0, p_x = p_y: hyperbolic point of Omega_(1,-1,0).  Averaging over the fast angles gives
    (x - y)'' = eps sin(x - y), i.e. exponent sqrt(eps): FLI ~ sqrt(eps) t.  Off resonance FLI ~ ln t."""
    eps, n, dt = 1e-3, 100000, 0.01
    g = orc.make_grid(48, 48)
    st = orc.init_shell(orc.State(48 * 48), g, 1.0, eps, 0)
    sel = [10 * 48 + 10, 30 * 48 + 30, 10 * 48 + 37, 7 * 48 + 20, 33 * 48 + 11]  # 3 on the diagonals, 2 off
    for k in sel:
        orc.integrate(st, n, dt, 100, k, k + 1, advance_clock=False)
    t = n * dt
    fli = st.acc[1]
    for k in sel[:3]:
        assert 0.8 * math.sqrt(eps) * t < fli[k] < 1.3 * math.sqrt(eps) * t, fli[k]
    for k in sel[3:]:
        assert math.log(t) - 1.5 < fli[k] < math.log(t) + 1.0, fli[k]
    assert np.max(st.acc[3, sel]) < 1e-11                     # energy conserved along the way


def test_paper_resonance_geometry():
    """W = (sqrt E, sqrt E, 0) lies on the three named resonance planes and on the shell."""
    g = golden()
    for E in (15.0, 400.0, 1.0):
        W = math.sqrt(E) * np.array(g["W_over_sqrtE"])
        for key in ("W_res_1", "W_res_2", "W_res_3"):
            assert abs(np.dot(g[key], W)) < 1e-12
        assert abs(np.dot(W, W) - 2 * E) < 1e-12
    assert g["tesla_resident"][0] == g["tesla_resident"][1] * g["tesla_resident"][2]


# ------------------------------------------------------------------ a5: indicator image (R13, R14)

def test_indicator_kinds_thresholds_and_masks(orc):
    """awo_indicator on a hand-made accumulator table (no integration, nothing from the CUDA path): FLI is
    plane 1, FTLE is plane 0 divided by t, DH is plane 3; CLASS is the STRICT comparison FLI > thr (R14);
    every trajectory that is not live (status 0 off-shell, 2 non-finite, 3 left the area) reads NaN in the
    float kinds and 255 in the class byte."""
    n = 8
    st = orc.State(n, tangent=True, wind=False)
    thr = math.log(1000.0) + 3.0                                  # R14 at t = 1000
    up, dn = np.nextafter(thr, np.inf), np.nextafter(thr, -np.inf)
    #                 k:    0     1    2    3     4      5     6     7
    st.acc[0, :n] = [250.0, -3.0, 1.5, 7.25, 99.0, 12.5, 0.0, 4.0]        # logsum
    st.acc[1, :n] = [thr, up, dn, 7.25, 99.0, 99.0, 99.0, -0.0]           # fli_max
    st.acc[2, :n] = 1.0                                                   # H0 (not an output)
    st.acc[3, :n] = [1e-12, 2e-12, 3e-12, 4e-12, 5e-12, 6e-12, 7e-12, 0.0]  # dH_max
    st.status[:] = [1, 1, 1, 1, 0, 2, 3, 1]
    st.t = 1000.0
    live = st.status == 1
    fli, ftle, dh = orc.indicator(st, 0), orc.indicator(st, 1), orc.indicator(st, 2)
    for img in (fli, ftle, dh):
        assert np.array_equal(np.isnan(img), ~live)              # NaN exactly on the non-live ones
    assert np.array_equal(fli[live], np.array([thr, up, dn, 7.25, -0.0]))
    assert np.array_equal(ftle[live], np.array([0.25, -0.003, 0.0015, 0.00725, 0.004]))   # logsum / 1000, hand values
    assert np.array_equal(dh[live], np.array([1e-12, 2e-12, 3e-12, 4e-12, 0.0]))          # plane 3, not 0, 1 or 2
    cls = orc.indicator(st, 3, thr)
    #  FLI == thr -> regular (strict >), one ulp above -> chaotic, one below -> regular, 7.25 < 9.9 -> regular
    assert cls.tolist() == [0, 1, 0, 0, 255, 255, 255, 0]
    assert cls.dtype == np.uint8
    # the threshold is the argument, not a constant: a lower one flips pixel 3 only among the live regular ones
    assert orc.indicator(st, 3, 7.0).tolist() == [1, 1, 1, 1, 255, 255, 255, 0]
    assert orc.indicator(st, 3, 7.25).tolist() == [1, 1, 1, 0, 255, 255, 255, 0]
    # FTLE uses the elapsed time of the state
    st.t = 500.0
    assert np.array_equal(orc.indicator(st, 1)[live], np.array([0.5, -0.006, 0.003, 0.0145, 0.008]))
    # planes are addressed with the pitch, not n
    st2 = orc.State(3, tangent=True, wind=False, pitch=64)
    st2.acc[1, :3], st2.status[:], st2.t = [1.0, 2.0, 3.0], 1, 1.0
    assert orc.indicator(st2, 0).tolist() == [1.0, 2.0, 3.0]


def test_indicator_on_an_integrated_orbit_matches_the_eps0_closed_form(orc):
    """End to end through awo_integrate + awo_indicator at eps = 0: FLI = sup_t ln|w(t)| with
    |w(t)|^2 = |dX0 + t dP0|^2 + |dP0|^2 in closed form; FTLE = ln|w(T)| / T; DH = 0 up to rounding; the class
    byte follows from comparing the closed form with thr."""
    n = 64
    st = orc.init_shell(orc.State(n), orc.make_grid(8, 8, angle_mode=1, tangent_mode=1), 1.0, 0.0, 11)
    w0 = st.w[:, :n].copy()
    orc.integrate(st, 2000, 0.01, 100)
    ts = 0.01 * 100 * np.arange(1, 21)
    norms = np.array([0.5 * np.log(((w0[:3] + t * w0[3:]) ** 2).sum(0) + (w0[3:] ** 2).sum(0)) for t in ts])
    ref_fli = np.maximum(norms.max(0), 0.0)
    assert np.max(np.abs(orc.indicator(st, 0) - ref_fli)) < 1e-12
    assert np.max(np.abs(orc.indicator(st, 1) - norms[-1] / 20.0)) < 1e-13
    assert orc.indicator(st, 2).max() < 1e-14
    thr = float(np.median(ref_fli))
    sure = np.abs(ref_fli - thr) > 1e-9
    assert np.array_equal(orc.indicator(st, 3, thr)[sure], (ref_fli > thr).astype(np.uint8)[sure])


# ------------------------------------------------------------------ slices of the ensemble (k0)

@pytest.mark.parametrize("shape,angle_mode,tmode", [(0, 0, 0), (0, 1, 1), (1, 1, 0), (2, 1, 1), (3, 1, 1)])
def test_init_shell_slices_are_rows_of_the_whole_ensemble(orc, shape, angle_mode, tmode):
    """P:13, P:63 (independent realisations): a state that holds trajectories [k0, k0 + n) of the ensemble is,
    bit for bit, that slice of the whole — grid position and every random draw are functions of the GLOBAL index.
    The grid values themselves are re-derived here from the definition (cell centres, R6)."""
    gx, gy = 12, 10
    E, eps, seed = 1.0, 2e-2, 5
    mk = lambda k0: orc.make_grid(gx, gy, -0.9, 0.7, angle_mode, shape, 0.1, -0.2, 0.05, 1, tmode,
                                  lo_y=-0.5, hi_y=0.8, k0=k0)
    whole = orc.init_shell(orc.State(gx * gy), mk(0), E, eps, seed)
    for k0, n in ((0, 37), (37, 50), (87, 33), (119, 1), (60, 0)):
        part = orc.init_shell(orc.State(n), mk(k0), E, eps, seed)
        assert np.array_equal(part.q[:, :n], whole.q[:, k0:k0 + n], equal_nan=True)
        assert np.array_equal(part.w[:, :n], whole.w[:, k0:k0 + n])
        assert np.array_equal(part.acc[:, :n], whole.acc[:, k0:k0 + n], equal_nan=True)
        assert np.array_equal(part.status, whole.status[k0:k0 + n])
        if shape == 0 and n:
            K = k0 + np.arange(n)
            px = -0.9 + ((K % gx) + 0.5) * (0.7 - -0.9) / gx
            py = -0.5 + ((K // gx) + 0.5) * (0.8 - -0.5) / gy
            assert np.array_equal(part.q[3, :n], px) and np.array_equal(part.q[4, :n], py)
        if angle_mode and n:
            assert part.q[0, 0] == 2 * math.pi * orc.uniform(seed, k0, 0) or np.isnan(part.q[0, 0])
    # a slice may not reach past the ensemble
    import ctypes
    bad = orc.State(5)
    g = mk(gx * gy - 4)
    rc = orc.lib().awo_init_shell(ctypes.byref(g), E, eps, seed, 5, bad.pitch, bad.q.ctypes.data_as(orc._dp),
                                  bad.w.ctypes.data_as(orc._dp), bad.acc.ctypes.data_as(orc._dp),
                                  bad.wind.ctypes.data_as(orc._i32p), bad.status.ctypes.data_as(orc._u8p))
    assert rc == -1


def test_gaussian_cloud_is_a_2d_normal(orc):
    """"Gaussian distribution ... with the dispersion sigma": the radius of a 2-d normal is Rayleigh,
    P(r < a sigma) = 1 - exp(-a^2/2); components independent with variance sigma^2; the centre is W."""
    n = 1 << 16
    sig, cx, cy = 0.01, math.sqrt(15.0), math.sqrt(15.0)
    g = orc.make_grid(256, 256, angle_mode=1, shape=2, cx=cx, cy=cy, r=sig)
    st = orc.init_shell(orc.State(n, tangent=False), g, 15.0, 1.0, 4)
    live = st.status == 1
    # W lies on the equator pz = 0 of the E = 15 shell: roughly half the cloud is outside the shell (R8)
    assert 0.3 < live.mean() < 0.7
    g2 = orc.make_grid(256, 256, angle_mode=1, shape=2, cx=1.0, cy=-2.0, r=sig)
    s2 = orc.init_shell(orc.State(n, tangent=False), g2, 15.0, 1.0, 4)
    assert np.all(s2.status == 1)
    dx, dy = s2.q[3, :n] - 1.0, s2.q[4, :n] + 2.0
    r = np.hypot(dx, dy) / sig
    for a in (0.5, 1.0, 2.0, 3.0):
        assert abs((r < a).mean() - (1 - math.exp(-a * a / 2))) < 4e-3
    assert abs(dx.std() / sig - 1) < 0.01 and abs(dy.std() / sig - 1) < 0.01
    assert abs(np.corrcoef(dx, dy)[0, 1]) < 0.012 and abs(dx.mean()) < 1.2e-4 and abs(dy.mean()) < 1.2e-4
    H = 0.5 * (s2.q[3:, :n] ** 2).sum(0) + np.cos(s2.q[0, :n]) * np.cos(s2.q[1, :n]) * (1 + np.cos(2 * s2.q[2, :n]))
    assert np.max(np.abs(H - 15.0)) < 64 * np.spacing(15.0)                 # v_z from the energy condition


def test_cloud_resampling_is_rejection_sampling(orc):
    """R31 (v_z "calculated from the fixed energy condition"; a draw without a real v_z is drawn again):
    attempt a takes every draw of the trajectory from seed + a * 0xD1B54A32D192ED03.  Pinned by re-deriving the
    accepted attempt from plain (resample = 0) ensembles generated with those seeds, and by the statistics: the
    accepted points are distributed like the on-shell points of the plain ensemble (same conditional law)."""
    n = 1 << 13
    W = math.sqrt(15.0)
    mk = lambda resample: orc.make_grid(128, 64, angle_mode=1, shape=2, cx=W, cy=W, r=0.01, resample=resample)
    plain = [orc.init_shell(orc.State(n, tangent=False), mk(0), 15.0, 1.0, (7 + a * 0xD1B54A32D192ED03) % 2 ** 64)
             for a in range(6)]
    res = orc.init_shell(orc.State(n, tangent=False), mk(5), 15.0, 1.0, 7)
    first = np.full(n, -1)
    for a in reversed(range(6)):
        first[plain[a].status == 1] = a
    assert 0.3 < (first == 0).mean() < 0.7 and (first == 1).sum() > 0 and (first == 5).sum() > 0
    assert np.array_equal(res.status == 1, first >= 0)
    for a in range(6):
        sel = first == a
        assert np.array_equal(res.q[:, :n][:, sel], plain[a].q[:, :n][:, sel])
        assert np.array_equal(res.acc[2, :n][sel], plain[a].acc[2, :n][sel])
    assert np.isnan(res.q[:, :n][:, first < 0]).all()
    # enough attempts: everyone is on the shell (P(all 40 draws fail) ~ 2^-40), H = E for all
    full = orc.init_shell(orc.State(n, tangent=False), mk(40), 15.0, 1.0, 7)
    assert np.all(full.status == 1) and np.max(np.abs(full.acc[2, :n] - 15.0)) < 64 * np.spacing(15.0)
    # same conditional law as the masked ensemble: compare the first two moments of (px, py) and of H_p
    big = orc.init_shell(orc.State(1 << 16, tangent=False), orc.make_grid(256, 256, angle_mode=1, shape=2, cx=W, cy=W,
                                                                         r=0.01), 15.0, 1.0, 99)
    lv = big.status == 1
    hp = lambda s, m: (np.cos(s.q[0, :s.n]) * np.cos(s.q[1, :s.n]) * (1 + np.cos(2 * s.q[2, :s.n])))[m]
    all_live = np.ones(n, bool)
    assert abs(hp(full, all_live).mean() - hp(big, lv).mean()) < 0.03           # both ~ E[H_p | on shell] < 0
    assert hp(full, all_live).max() < 0.3 and hp(big, lv).mean() < -0.3      # 2 H_p <= 2E - px^2 - py^2 ~ +-0.1
    assert abs(full.q[3, :n].mean() - big.q[3, :big.n][lv].mean()) < 5e-4
    assert abs(full.q[3, :n].std() - big.q[3, :big.n][lv].std()) < 5e-4
    # grids and the sphere ignore the flag
    for shape in (0, 3):
        a_ = orc.init_shell(orc.State(64, tangent=False), orc.make_grid(8, 8, angle_mode=1, shape=shape, resample=0), 1.0, 3e-2, 1)
        b_ = orc.init_shell(orc.State(64, tangent=False), orc.make_grid(8, 8, angle_mode=1, shape=shape, resample=9), 1.0, 3e-2, 1)
        assert np.array_equal(a_.q, b_.q, equal_nan=True)


def test_random_rectangle_patch(orc):
    """R33 ("uniformly distributed within a small segment of the sphere (enclosed by the two squares ...)"):
    shape 4 draws (px, py) uniformly at random in [lo_x, hi_x) x [lo_y, hi_y): px = lo_x + u3 (hi_x - lo_x) with the
    generator's own draws (retyped here), uniform by chi-square, v_z from the energy condition, angles uniform."""
    n = 1 << 14
    lo_x, hi_x, lo_y, hi_y = 1.0, 1.5, -2.25, -2.0
    g = orc.make_grid(128, 128, lo_x, hi_x, angle_mode=1, shape=4, lo_y=lo_y, hi_y=hi_y)
    st = orc.init_shell(orc.State(n, tangent=False), g, 15.0, 1.0, 21)
    assert np.all(st.status == 1)                                   # well inside the E = 15 shell: P^2 <= 7.3 < 26
    u3 = np.array([orc.uniform(21, k, 3) for k in range(n)])
    u4 = np.array([orc.uniform(21, k, 4) for k in range(n)])
    assert np.array_equal(st.q[3, :n], lo_x + u3 * (hi_x - lo_x)) and np.array_equal(st.q[4, :n], lo_y + u4 * (hi_y - lo_y))
    assert st.q[3, :n].min() >= lo_x and st.q[3, :n].max() < hi_x and st.q[4, :n].min() >= lo_y and st.q[4, :n].max() < hi_y
    counts = np.histogram2d(st.q[3, :n], st.q[4, :n], bins=8, range=((lo_x, hi_x), (lo_y, hi_y)))[0].ravel()
    assert ((counts - n / 64) ** 2 / (n / 64)).sum() < 120          # 63 dof: mean 63, sd 11
    assert abs(np.corrcoef(st.q[3, :n], st.q[4, :n])[0, 1]) < 0.03
    H = 0.5 * (st.q[3:, :n] ** 2).sum(0) + np.cos(st.q[0, :n]) * np.cos(st.q[1, :n]) * (1 + np.cos(2 * st.q[2, :n]))
    assert np.max(np.abs(H - 15.0)) < 64 * np.spacing(15.0) and np.all(st.q[5, :n] > 0)
    # a patch that reaches over the edge of the shell: masked, or drawn again with resample (R31)
    g2 = orc.make_grid(64, 64, 3.6, 4.0, angle_mode=1, shape=4, lo_y=3.6, hi_y=4.0)
    s2 = orc.init_shell(orc.State(4096, tangent=False), g2, 15.0, 1.0, 21)
    assert 0 < (s2.status == 0).sum() < 4096
    g3 = orc.make_grid(64, 64, 3.6, 4.0, angle_mode=1, shape=4, lo_y=3.6, hi_y=4.0, resample=60)
    s3 = orc.init_shell(orc.State(4096, tangent=False), g3, 15.0, 1.0, 21)
    assert np.all(s3.status == 1)
    first = s2.status == 1
    assert np.array_equal(s3.q[:, :4096][:, first], s2.q[:, :4096][:, first])

"""GPU parity tests (-m gpu) added in round 2, each through the C ABI against the oracle on the same seeded inputs:

  * Gaussian-cloud initial conditions (shape 2) against the oracle's generator;
  * the Fig. 4 workload: cloud at W, density of the projected averaged velocity accumulated
    over CONSECUTIVE averaging windows;
  * the energy bound of the trigonometry level is enforced on the device, not assumed (aw_state.Emax, AW_ST_RANGE,
    aw_bound_energy, aw_map_host picks the level from the uploaded data);
  * slices [k0, k0 + n) of an ensemble are bit-identical to the same rows of the whole (multi-GPU sharding);
  * the integrator's block size does not change a bit of the result;
  * odd histogram sizes with dropped points (64-bit drop counter alignment).

Bars as in test_gpu_parity.py (BASELINE north_star): state 1e-10 relative at <= 1000 steps for regular orbits, 100
steps for all; integer work bit-exact.
"""
import math

import numpy as np
import pytest
import torch

from util import ensemble_to_oracle, oracle_integrate_mt, state_rel_err

pytestmark = pytest.mark.gpu

ULP1 = 2.0 ** -52


@pytest.fixture(scope="module")
def aw():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1107_4107_b200 import build
    build.build()
    import paper_1107_4107_b200 as aw
    return aw


# ------------------------------------------------------------------ table-driven sincos of the step loop

def test_table_sincos_within_2ulp(aw):
    """csrc/aw_tsincos.cuh (DESIGN.md §6.1 (ii)) against libm / mpmath on 5e6 random points of the range the integrator
    produces (|x| < 1024, R7), every table grid point and the midpoints between them: <= 2 ulp of max(|result|, s1)
    with s1 = sin(2 pi / 512) = 0.0123 — the statement pin P14 makes for the device sincos wherever |result| >= s1, and
    an absolute 3.5e-18 nearer a zero of the function, where the result is the difference of a table entry and a
    correction of the same size (the kick multiplies it by O(1) factors: what matters there is the error relative to
    the amplitude, 0.016 ulp).  Exact at 0, sin bit-odd and cos bit-even."""
    import aw_probe
    rng = np.random.default_rng(41)
    grid = np.arange(-2048, 2049) * (2 * math.pi / 512)
    x = np.concatenate([rng.uniform(-16 * math.pi, 16 * math.pi, 4_000_000), rng.uniform(-1024.0, 1024.0, 1_000_000),
                        rng.uniform(-1e-3, 1e-3, 100_000), grid, grid + math.pi / 512,
                        np.array([0.0, -0.0, math.pi, -math.pi, math.pi / 2, 1e-300, 5e-324])])
    s, c = aw_probe.tsincos(torch.from_numpy(x).cuda())
    s, c = s.cpu().numpy(), c.cpu().numpy()
    rs, rc = np.sin(x), np.cos(x)

    s1 = math.sin(2 * math.pi / 512)
    floor_ulp = np.spacing(s1)

    def excess(a, b):
        return np.abs(a - b) - 2.0 * np.maximum(np.spacing(np.abs(b)), floor_ulp)
    assert excess(s, rs).max() <= 0.0, excess(s, rs).max()
    assert excess(c, rc).max() <= 0.0, excess(c, rc).max()
    nr = 5_100_000
    ulps = lambda a, b: np.abs(a - b) / np.maximum(np.spacing(np.abs(b)), floor_ulp)
    assert ulps(s[:nr], rs[:nr]).max() <= 2.0 and ulps(c[:nr], rc[:nr]).max() <= 2.0
    import mpmath as mp
    mp.mp.dps = 40
    for i in rng.integers(0, nr, 2000):
        xs = mp.mpf(float(x[i]))
        es = abs(mp.mpf(float(s[i])) - mp.sin(xs)) / mp.mpf(float(max(np.spacing(abs(rs[i])), floor_ulp)))
        ec = abs(mp.mpf(float(c[i])) - mp.cos(xs)) / mp.mpf(float(max(np.spacing(abs(rc[i])), floor_ulp)))
        assert es <= 1.6 and ec <= 1.6, (x[i], es, ec)
    s0, c0 = aw_probe.tsincos(torch.zeros(1, dtype=torch.float64, device="cuda"))
    assert s0.item() == 0.0 and c0.item() == 1.0
    sm, cm = aw_probe.tsincos(torch.from_numpy(-x).cuda())
    assert np.array_equal(sm.cpu().numpy(), -s) and np.array_equal(cm.cpu().numpy(), c)
    # agreement with the device sincos the checkpoints use: both within 2 ulp of the truth
    sd, cd = aw_probe.sincos(torch.from_numpy(x[:nr]).cuda())
    assert ulps(s[:nr], sd.cpu().numpy()).max() <= 4.0 and ulps(c[:nr], cd.cpu().numpy()).max() <= 4.0


# ------------------------------------------------------------------ P:97 Gaussian cloud (shape 2)

@pytest.mark.parametrize("E,eps,cx,cy,sigma,pz_sign", [
    (15.0, 1.0, math.sqrt(15.0), math.sqrt(15.0), 0.01, 1),     # the paper's cloud at W: on the equator, ~half masked
    (1.0, 3e-2, 0.99, 0.98, 0.02, -1),                          # near the equator of the E = 1 shell, lower hemisphere
    (1.0, 1e-3, 0.1, -0.2, 0.01, 1)])                           # well inside: nobody masked
def test_gauss_init_matches_oracle_generator(aw, orc, E, eps, cx, cy, sigma, pz_sign):
    gx, gy = 131, 67                                            # ragged: 8777 trajectories
    n = gx * gy
    for tmode in (0, 1):
        ens = aw.Ensemble(n, tangent=True, wind=True)
        aw.aw_init_shell(ens, aw.make_grid(gx, gy, angle_mode=1, shape=aw.AW_SHAPE_GAUSS, cx=cx, cy=cy, r=sigma,
                                           pz_sign=pz_sign, tangent_mode=tmode), E, eps, 97)
        ref = orc.State(n, True, True)
        orc.init_shell(ref, orc.make_grid(gx, gy, angle_mode=1, shape=2, cx=cx, cy=cy, r=sigma, pz_sign=pz_sign,
                                          tangent_mode=tmode), E, eps, 97)
        got = ensemble_to_oracle(ens, orc)
        # The mask is the sign of the radicand R = 2(E - eps H_p) - px^2 - py^2, which both sides round separately
        # (libm vs device cos, log, sqrt: <= 1 ulp each): decisions agree except where |R| is at the rounding level
        differ = got.status != ref.status
        live = (got.status == 1) & (ref.status == 1)
        assert differ.sum() <= 2
        if cx > 0.5:
            assert 0 < (ref.status == 0).sum() < n               # some points are off the shell (R8)
        else:
            assert np.all(ref.status == 1)
        assert np.array_equal(got.q[:3, :n][:, live], ref.q[:3, :n][:, live])      # angles: integer hash * constant
        scale = math.sqrt(2 * (E + 2 * eps))
        # px, py: centre + sigma * Box-Muller (log, sqrt, sincos differ by <= 1 ulp each between libm and the device)
        assert np.max(np.abs(got.q[3:5, :n][:, live] - ref.q[3:5, :n][:, live])) <= 4e-15 * scale
        # pz = sqrt(R): the cancellation in R amplifies the rounding of px, py by |p|/pz; compare pz^2
        dpz2 = np.abs(got.q[5, :n][live] ** 2 - ref.q[5, :n][live] ** 2)
        assert np.max(dpz2) <= 64 * ULP1 * scale ** 2
        assert np.all(np.sign(got.q[5, :n][live]) * pz_sign >= 0)
        assert np.isnan(got.q[:, :n][:, got.status == 0]).all() and np.isnan(got.acc[2, :n][got.status == 0]).all()
        assert np.max(np.abs(got.acc[2, :n][live] - E)) <= 16 * np.spacing(E)        # H0 = E (v_z from the energy)
        assert np.all(got.acc[[0, 1, 3], :n] == 0.0) and np.all(got.wind == 0)
        assert np.allclose(got.w[:, :n], ref.w[:, :n], rtol=0, atol=2e-15)


@pytest.mark.parametrize("shape,resample", [(2, 3), (2, 40), (1, 5)])
def test_cloud_resampling_matches_oracle_generator(aw, orc, shape, resample):
    """R31: draws without a real v_z are drawn again from the attempt seeds; the device generator accepts the same
    attempt as the oracle's for every trajectory (up to a radicand at the rounding level), k0 slices included."""
    W = math.sqrt(15.0)
    gx, gy, k0 = 97, 61, 1000
    n = gx * gy - k0 - 7
    mk = lambda mod: mod.make_grid(gx, gy, angle_mode=1, shape=shape, cx=W, cy=W, r=0.01 if shape == 2 else 0.02,
                                   k0=k0, resample=resample)
    ens = aw.Ensemble(n, tangent=False, wind=True)
    aw.aw_init_shell(ens, mk(aw), 15.0, 1.0, 31)
    ref = orc.init_shell(orc.State(n, tangent=False), mk(orc), 15.0, 1.0, 31)
    got = ensemble_to_oracle(ens, orc)
    both = (got.status == 1) & (ref.status == 1)
    same = both & np.all(got.q[:3, :n] == ref.q[:3, :n], axis=0)
    assert (got.status != ref.status).sum() + (both & ~same).sum() <= 2
    if resample == 40:
        assert np.all(ref.status == 1) and np.all(got.status == 1)
    else:
        assert 0 < (ref.status == 0).sum() < 0.2 * n              # P(off shell)^(resample + 1) of the draws remain masked
    assert np.max(np.abs(got.q[3:5, :n][:, same] - ref.q[3:5, :n][:, same])) <= 4e-14
    assert np.max(np.abs(got.q[5, :n][same] ** 2 - ref.q[5, :n][same] ** 2)) <= 64 * ULP1 * 34.0
    assert np.max(np.abs(got.acc[2, :n][got.status == 1] - 15.0)) <= 16 * np.spacing(15.0)
    bad = mk(aw)
    bad.resample = -1
    with pytest.raises(aw.AwError):
        aw.aw_init_shell(ens, bad, 15.0, 1.0, 31)


# ------------------------------------------------------------------ P:87 / P:99: random square segment, survivors

def test_zoom_square_with_survivors_parity(aw, orc):
    """CONFIGS[9] at reduced size: initial conditions uniformly at random in a square segment of the sphere (shape
    RECT), survivor filter on the launch square, window Dt = 100 T.  Generator bit-equal to the
    oracle's (px, py are hash * constant arithmetic); after 100 steps every state within 1e-10; after the window the
    survivor statuses equal the oracle's except where (px, py) passes within rounding distance of an edge, and the
    sphere density of the survivors is bit-exact on the device states."""
    cfg = aw.CONFIGS[9]
    gx, gy = 96, 64
    n = gx * gy
    rect = (cfg["lo"], cfg["hi"], cfg["lo"], cfg["hi"])
    mk = lambda mod: mod.make_grid(gx, gy, cfg["lo"], cfg["hi"], cfg["angle_mode"], cfg["shape"])
    ens = aw.Ensemble(n, tangent=False, wind=True, order=cfg["order"], ref=True)
    aw.aw_init_shell(ens, mk(aw), cfg["E"], cfg["eps"], cfg["seed"])
    gen = orc.init_shell(orc.State(n, tangent=False), mk(orc), cfg["E"], cfg["eps"], cfg["seed"])
    st = ensemble_to_oracle(ens, orc)
    assert np.all(st.status == 1) and np.array_equal(st.status, gen.status)
    assert np.array_equal(st.q[:5, :n], gen.q[:5, :n])                        # angles, px, py: bit-equal
    assert np.max(np.abs(st.q[5, :n] - gen.q[5, :n])) <= 4e-15 * math.sqrt(34.0)
    ens.set_survivors(rect)
    aw.aw_mark(ens)
    st = ensemble_to_oracle(ens, orc)
    aw.aw_integrate(ens, n, 100, cfg["dt"], cfg["stride"])
    orc.integrate(st, 100, cfg["dt"], cfg["stride"])
    got = ensemble_to_oracle(ens, orc)
    assert np.array_equal(got.status, st.status)
    err = state_rel_err(got.q[:, :n], got.wind[:, :n], st.q[:, :n], st.wind[:, :n], np.ones(n, bool))
    assert err.max() <= 1e-10, err.max()
    aw.aw_integrate(ens, n, cfg["steps"] - 100, cfg["dt"], cfg["stride"])
    oracle_integrate_mt(orc, st, cfg["steps"] - 100, cfg["dt"], cfg["stride"])
    got = ensemble_to_oracle(ens, orc)
    gone = st.status == 3
    assert 0.2 * n < gone.sum() < n                                            # a chaotic neighbourhood: many leave
    # decisions differ only for trajectories that graze an edge of the square (chaotic orbits decorrelate over 100 T)
    assert (got.status != st.status).sum() <= 0.02 * n
    assert abs((ens.t - ens.tref) - 100 * 2 * math.pi) < 1e-8
    G = 128
    hist = torch.zeros((G, G), dtype=torch.int32, device="cuda")
    dropped = torch.zeros(1, dtype=torch.int64, device="cuda")
    aw.aw_density(ens, hist, cfg["hist_lo"], cfg["hist_hi"], cfg["density_mode"], dropped)
    ref = np.zeros((G, G), dtype=np.uint32)
    d = orc.density_velocity(got, ref, cfg["hist_lo"], cfg["hist_hi"], cfg["density_mode"])
    h = hist.cpu().numpy().view(np.uint32)
    assert np.array_equal(h, ref) and int(dropped.item()) == int(d[0])
    assert int(h.sum()) + int(d[0]) == int((got.status == 1).sum())
    assert h.sum() > 0


# ------------------------------------------------------------------ P:97 Fig. 4: consecutive windows

def test_fig4_consecutive_windows_density_parity(aw, orc):
    """CONFIGS[7] (N = 3.2e4 trajectories in a Gaussian cloud at W, resampled onto the shell, E = 15, eps = 1, order 6, h = 0.01 T) in the
    launch configuration bench.py --config 7 times: windows x (aw_mark; aw_integrate(Dt = 50 T); aw_density mode 3
    ACCUMULATING) = the density "averaged over the whole time span between consecutive plots".  After each of
    three consecutive windows the accumulated histogram is bit-exact against the oracle's binning of the device
    states; sampled state parity after the first 100 steps; P:51 shell layer and energy at the end."""
    cfg = aw.CONFIGS[7]
    n = cfg["gx"] * cfg["gy"]
    ens = aw.Ensemble(n, tangent=False, wind=True, order=cfg["order"], ref=True)
    g = aw.make_grid(cfg["gx"], cfg["gy"], cfg["lo"], cfg["hi"], cfg["angle_mode"], cfg["shape"], cfg["cx"], cfg["cy"],
                     cfg["r"], resample=cfg["resample"])
    aw.aw_init_shell(ens, g, cfg["E"], cfg["eps"], cfg["seed"])
    assert aw.aw_trig_level(ens, cfg["dt"]) == 7
    st0 = ensemble_to_oracle(ens, orc)
    live0 = st0.status == 1
    assert n == 32_000 and live0.all()                          # the paper's N = 3.2e4, every draw on the shell
    # the generator with resampling (R31) against the oracle's: same accepted attempt for every trajectory
    gen = orc.init_shell(orc.State(n, tangent=False), orc.make_grid(cfg["gx"], cfg["gy"], cfg["lo"], cfg["hi"],
                         cfg["angle_mode"], cfg["shape"], cfg["cx"], cfg["cy"], cfg["r"], resample=cfg["resample"]),
                         cfg["E"], cfg["eps"], cfg["seed"])
    assert np.all(gen.status == 1)
    same = np.all(gen.q[:3, :n] == st0.q[:3, :n], axis=0)        # angles are hash * constant: equal iff same attempt
    assert (~same).sum() <= 2                                    # radicand at the rounding level may flip an attempt
    assert np.max(np.abs(gen.q[3:5, :n][:, same] - st0.q[3:5, :n][:, same])) <= 4e-14
    # state parity, 100 steps, on 512 sampled live trajectories (the region around W is strongly chaotic)
    sample = np.nonzero(live0)[0][:: max(1, int(live0.sum()) // 512)][:512]
    probe = aw.Ensemble(n, tangent=False, wind=True, order=cfg["order"])
    aw.aw_init_shell(probe, g, cfg["E"], cfg["eps"], cfg["seed"])
    aw.aw_integrate(probe, n, 100, cfg["dt"], cfg["stride"])
    for k in sample:
        orc.integrate(st0, 100, cfg["dt"], cfg["stride"], k0=int(k), k1=int(k) + 1, advance_clock=False)
    got = ensemble_to_oracle(probe, orc)
    err = state_rel_err(got.q[:, sample], got.wind[:, sample], st0.q[:, sample], st0.wind[:, sample],
                        np.ones(len(sample), bool))
    assert err.max() <= 1e-10, err.max()
    # three consecutive windows, accumulated density
    G, lo, hi = 512, cfg["hist_lo"], cfg["hist_hi"]
    hist = torch.zeros((G, G), dtype=torch.int32, device="cuda")
    dropped = torch.zeros(1, dtype=torch.int64, device="cuda")
    ref = np.zeros((G, G), dtype=np.uint32)
    d = np.zeros(1, dtype=np.uint64)
    per_window = []
    for wdw in range(3):
        aw.aw_mark(ens)
        assert ens.tref == ens.t
        aw.aw_integrate(ens, n, cfg["window"], cfg["dt"], cfg["stride"])
        assert abs((ens.t - ens.tref) - 50 * 2 * math.pi) < 1e-9
        aw.aw_density(ens, hist, lo, hi, cfg["density_mode"], dropped)
        dev = ensemble_to_oracle(ens, orc)
        assert dev.tref == ens.tref and np.array_equal(dev.status == 1, live0)
        before = ref.copy()
        orc.density_velocity(dev, ref, lo, hi, cfg["density_mode"], d)
        per_window.append(ref - before)
        h = hist.cpu().numpy().view(np.uint32)
        assert np.array_equal(h, ref) and int(dropped.item()) == int(d[0])
        assert int(h.sum()) + int(d[0]) == (wdw + 1) * int(live0.sum())
    # the windows are different windows (the snapshot moved), and the cloud spreads away from W
    assert not np.array_equal(per_window[0], per_window[1]) and not np.array_equal(per_window[1], per_window[2])
    occupied = [(p > 0).sum() for p in per_window]
    assert occupied[2] > occupied[0]
    # energy conserved by the sixth-order scheme over 150 T (~1e-6 at E = 15), shell layer P:51
    P2 = (dev.q[3:, :n][:, live0] ** 2).sum(0)
    assert dev.acc[3, :n][live0].max() < 1e-5
    assert np.all(P2 >= 2 * (15.0 - 2.0) - 1e-4) and np.all(P2 <= 2 * (15.0 + 2.0) + 1e-4)


# ------------------------------------------------------------------ the energy bound is enforced (aw_state.Emax)

def _hot_states(orc, n, pitch, eps, pnorm_hi, seed=21):
    """n hand-made states: random angles and directions; the first half with |P| = sqrt(2), the second half with
    |P| = pnorm_hi (test-side arithmetic, no oracle or library call except H0)."""
    rng = np.random.default_rng(seed)
    q = np.zeros((6, pitch))
    q[:3, :n] = rng.uniform(-math.pi, math.pi, (3, n))
    d = rng.normal(size=(3, n))
    d /= np.linalg.norm(d, axis=0)
    pn = np.where(np.arange(n) < n // 2, math.sqrt(2.0), pnorm_hi)
    q[3:, :n] = d * pn
    acc = np.zeros((4, pitch))
    acc[2, :n] = [orc.hamiltonian(q[:, k], eps) for k in range(n)]
    w = np.zeros((6, pitch))
    w[:, :n] = rng.normal(size=(6, n))
    w[:, :n] /= np.linalg.norm(w[:, :n], axis=0)
    return q, w, acc


def test_energy_bound_is_enforced_not_assumed(aw, orc):
    """The rotation kernels' Taylor degrees are sized for |P| <= sqrt(2(Emax + 2|eps|)).  Uploaded states with |P|
    three times the struct's bound: (a) aw_integrate flags them AW_ST_RANGE and leaves them untouched, bit for bit,
    while the trajectories inside the bound integrate normally; (b) after aw_bound_energy the same call integrates
    everyone and matches the oracle to 1e-10; (c) aw_map_host picks the level from the data by itself."""
    n, eps, dt = 2048 + 37, 3e-2, 0.005
    bound = math.sqrt(2 * (1.0 + 2 * eps))
    pitch = (n + 31) // 32 * 32
    q, w, acc = _hot_states(orc, n, pitch, eps, 3.0 * bound)
    status = np.ones(n, dtype=np.uint8)
    wind = np.zeros((3, pitch), dtype=np.int32)
    hot = np.arange(n) >= n // 2

    ref = orc.State(n, True, True)
    ref.q[:], ref.w[:], ref.acc[:], ref.status[:] = q, w, acc, status
    ref.E, ref.eps, ref.order = 1.0, eps, 4
    oracle_integrate_mt(orc, ref, 1000, dt, 100)
    thr = math.log(ref.t) + 3.0
    regular = ref.acc[1, :n] <= thr
    assert regular[hot].sum() > 0.8 * hot.sum()

    # (a) struct says E = 1: level 1, sized for |P| <= 1.456 (+ the level's slack); the hot half is flagged
    ens = aw.Ensemble(n, tangent=True, wind=True)
    ens.load_host(q, w, acc, wind, status, 1.0, eps)
    assert aw.aw_trig_level(ens, dt) == 1
    aw.aw_integrate(ens, n, 1000, dt, 100)
    got = ensemble_to_oracle(ens, orc)
    assert np.all(got.status[hot] == aw.AW_ST_RANGE) and np.all(got.status[~hot] == 1)
    assert np.array_equal(got.q[:, :n][:, hot], q[:, :n][:, hot]) and np.array_equal(got.w[:, :n][:, hot], w[:, :n][:, hot])
    assert np.array_equal(got.acc[:, :n][:, hot], acc[:, :n][:, hot])
    cool = ~hot & regular
    err = state_rel_err(got.q[:, :n], got.wind[:, :n], ref.q[:, :n], ref.wind[:, :n], cool)
    assert err.max() <= 1e-10, err.max()
    fli = aw.aw_indicator(ens, aw.AW_IND_FLI).cpu().numpy()
    assert np.isnan(fli[hot]).all() and np.isfinite(fli[~hot]).all()       # flagged pixels are masked, not wrong

    # (b) bound from the data, then the same call
    ens = aw.Ensemble(n, tangent=True, wind=True)
    ens.load_host(q, w, acc, wind, status, 1.0, eps)
    emax = aw.aw_bound_energy(ens)
    assert abs(emax - acc[2, :n].max()) <= 8 * np.spacing(emax) and ens.Emax == emax
    assert aw.aw_trig_level(ens, dt) >= 3
    aw.aw_integrate(ens, n, 1000, dt, 100)
    got = ensemble_to_oracle(ens, orc)
    assert np.all(got.status == 1)
    err = state_rel_err(got.q[:, :n], got.wind[:, :n], ref.q[:, :n], ref.wind[:, :n], regular)
    assert err.max() <= 1e-10, err.max()
    lo10 = ref.acc[1, :n] < 10
    assert np.max(np.abs(got.acc[1, :n][lo10] - ref.acc[1, :n][lo10])) <= 1e-5

    # (c) aw_map_host: host buffers in, struct still says E = 1
    b = aw.Ensemble(n, tangent=True, wind=True)
    b.c.E, b.c.eps = 1.0, eps
    host_in = dict(q=torch.from_numpy(q).pin_memory(), w=torch.from_numpy(w).pin_memory(),
                   acc=torch.from_numpy(acc).pin_memory(), wind=torch.from_numpy(wind).pin_memory(),
                   status=torch.from_numpy(status).pin_memory())
    out = dict(image=torch.empty(n, dtype=torch.float64).pin_memory(),
               q=torch.empty((6, pitch), dtype=torch.float64).pin_memory(),
               status=torch.empty(n, dtype=torch.uint8).pin_memory())
    ind_dev = torch.empty(n, dtype=torch.float64, device="cuda")
    aw.aw_map_host(b, host_in, 1000, dt, 100, aw.AW_IND_FLI, 0.0, (8, 8), -1.0, 1.0, ind_dev, None, out)
    assert bool((out["status"] == 1).all()) and b.Emax >= acc[2, :n].max() - 1e-12
    qh = out["q"].numpy()
    wh = b.wind.cpu().numpy()
    err = state_rel_err(qh[:, :n], wh[:, :n], ref.q[:, :n], ref.wind[:, :n], regular)
    assert err.max() <= 1e-10, err.max()
    assert np.max(np.abs(out["image"].numpy()[lo10] - ref.acc[1, :n][lo10])) <= 1e-5
    assert torch.equal(out["q"], ens.q.cpu())                    # same level, same kernel as (b): bit-identical

    # (d) the angle range of R7 is part of the same bound (level 0 has no Taylor limit, only the range of the
    # two-constant argument reduction): a stride the struct's E allows but the data does not
    c = aw.Ensemble(n, tangent=False, wind=True)
    c.load_host(q, None, acc, wind, status, 1.0, eps)
    c.trig = 1
    aw.aw_integrate(c, n, 600, 0.9, 600)                         # 600 * 0.9 * 1.456 < 1024 <= 600 * 0.9 * 4.37
    sc = c.status[:n].cpu().numpy()
    assert np.all(sc[hot] == aw.AW_ST_RANGE) and np.all(sc[~hot] == 1)
    c.status[:n] = 1                                             # the bound is taken over the LIVE trajectories
    aw.aw_bound_energy(c)
    with pytest.raises(aw.AwError) as ei:
        aw.aw_integrate(c, n, 600, 0.9, 600)
    assert ei.value.code == -3                                   # AW_ERANGE, refused on the host now


def test_bound_energy_edge_cases(aw):
    e0 = aw.Ensemble(0, tangent=False, wind=False)
    e0.c.E, e0.c.eps, e0.c.ready = 1.0, 1e-2, 1
    aw.aw_bound_energy(e0)
    # nobody live: Emax unchanged; NaN / inf states are ignored by the bound (the checkpoint flags them)
    n = 40
    ens = aw.Ensemble(n, tangent=False, wind=False)
    q = np.zeros((6, ens.pitch)); q[3, :n] = np.linspace(0.1, 2.0, n)
    q[3, 7] = np.inf; q[0, 9] = np.nan
    st = np.zeros(n, dtype=np.uint8)
    ens.load_host(q, None, np.zeros((4, ens.pitch)), None, st, 1.0, 0.0)
    assert aw.aw_bound_energy(ens) == 1.0
    st[:] = 1
    ens.load_host(q, None, np.zeros((4, ens.pitch)), None, st, 1.0, 0.0)
    assert aw.aw_bound_energy(ens) == 2.0                        # max finite P^2/2 at eps = 0
    q[3, :n] = -np.linspace(0.1, 0.5, n)
    ens.load_host(q, None, np.zeros((4, ens.pitch)), None, st, 1.0, 0.0)
    assert aw.aw_bound_energy(ens) == 0.125 and aw.aw_trig_level(ens, 0.005) == 1   # below E: E decides


# ------------------------------------------------------------------ slices of the ensemble (aw_grid.k0)

@pytest.mark.parametrize("shape,angle_mode,tmode", [(0, 0, 0), (0, 1, 1), (1, 1, 0), (2, 1, 1), (3, 1, 1)])
def test_slices_are_bit_identical_to_the_whole(aw, orc, shape, angle_mode, tmode):
    """a rank that holds trajectories [k0, k0 + n) of the ensemble computes, bit for bit, those rows of
    the single-GPU result — initial conditions (grid position and random draws are functions of the global index),
    integration, FLI image; the slices' histograms sum to the whole ensemble's."""
    gx, gy = 96, 41
    E, eps, seed = (15.0, 1.0, 8) if shape in (2, 3) else (1.0, 3e-2, 8)
    cx, cy, r = (3.0, 2.0, 0.05) if shape == 2 else (0.2, -0.1, 0.3)
    mk = lambda mod, k0: mod.make_grid(gx, gy, -0.9, 0.8, angle_mode, shape, cx, cy, r, 1, tmode, lo_y=-0.7, hi_y=0.9,
                                       k0=k0)
    n = gx * gy
    whole = aw.Ensemble(n, tangent=True, wind=True)
    aw.aw_init_shell(whole, mk(aw, 0), E, eps, seed)
    dt = 0.005 if E == 1.0 else 0.02
    aw.aw_integrate(whole, n, 300, dt, 100)
    fli = aw.aw_indicator(whole, aw.AW_IND_FLI)
    lim = math.sqrt(2 * E) * 1.1
    hw = torch.zeros((64, 64), dtype=torch.int32, device="cuda")
    aw.aw_density(whole, hw, -lim, lim)
    hs = torch.zeros((64, 64), dtype=torch.int32, device="cuda")
    cuts = [0, 7 * gx, 7 * gx + 13, 20 * gx, n - 1, n]           # whole rows, a ragged cut, a single trajectory
    for k0, k1 in zip(cuts[:-1], cuts[1:]):
        m = k1 - k0
        part = aw.Ensemble(m, tangent=True, wind=True)
        aw.aw_init_shell(part, mk(aw, k0), E, eps, seed)
        ref = orc.init_shell(orc.State(m), mk(orc, k0), E, eps, seed)          # the oracle's slice generator
        assert np.array_equal(part.status[:m].cpu().numpy(), ref.status)
        aw.aw_integrate(part, m, 300, dt, 100)
        assert np.array_equal(part.q[:, :m].cpu().numpy(), whole.q[:, k0:k1].cpu().numpy(), equal_nan=True)
        assert torch.equal(part.w[:, :m], whole.w[:, k0:k1]) and torch.equal(part.wind[:, :m], whole.wind[:, k0:k1])
        assert torch.equal(part.status[:m], whole.status[k0:k1])
        assert np.array_equal(aw.aw_indicator(part, aw.AW_IND_FLI).cpu().numpy(), fli[k0:k1].cpu().numpy(),
                              equal_nan=True)
        aw.aw_density(part, hs, -lim, lim)
    assert torch.equal(hs, hw)
    with pytest.raises(aw.AwError):
        aw.aw_init_shell(aw.Ensemble(5, tangent=False, wind=False), mk(aw, n - 4), E, eps, seed)


# ------------------------------------------------------------------ negative perturbation strength

@pytest.mark.parametrize("order,dt", [(4, 0.005), (6, 0.02), (4, 0.1), (6, 0.4)])
def test_negative_eps_parity(aw, orc, order, dt):
    """eps < 0 is a legal model (E - 2|eps| > 0): every stage weight b_s changes sign, and with it the factor 2 b_0 the
    kernel scales its carried zeta pair by.  Rotation and table kernels, tangent map on."""
    gx, gy = 67, 33
    n = gx * gy
    ens = aw.Ensemble(n, tangent=True, wind=True, order=order)
    aw.aw_init_shell(ens, aw.make_grid(gx, gy, -1.0, 1.0, angle_mode=1), 1.0, -3e-2, 13)
    st = ensemble_to_oracle(ens, orc)
    steps = 1000 if dt < 0.1 else 200
    aw.aw_integrate(ens, n, steps, dt, 100)
    oracle_integrate_mt(orc, st, steps, dt, 100)
    got = ensemble_to_oracle(ens, orc)
    assert np.array_equal(got.status, st.status)
    live = st.status == 1
    thr = math.log(st.t) + 3.0
    regular = live & (st.acc[1, :n] <= thr)
    assert regular.sum() > 0.5 * live.sum()
    err = state_rel_err(got.q[:, :n], got.wind[:, :n], st.q[:, :n], st.wind[:, :n], regular)
    assert err.max() <= 1e-10, err.max()
    lo10 = live & (st.acc[1, :n] < 10)
    assert np.max(np.abs(got.acc[1, :n][lo10] - st.acc[1, :n][lo10])) <= 1e-5
    P2 = (got.q[3:, :n][:, live] ** 2).sum(0)
    assert np.all(np.abs(P2 - 2.0) <= 4 * 3e-2 + 1e-6)                     # shell layer


# ------------------------------------------------------------------ block size

@pytest.mark.parametrize("order,tangent,dt", [(4, True, 0.005), (6, False, 0.0628), (6, True, 0.3), (4, False, 1.2)])
def test_block_size_does_not_change_the_result(aw, order, tangent, dt):
    """The integrator picks 32-, 64- or 128-thread blocks from n so that small ensembles spread over all SMs; the
    arithmetic is per trajectory, so every choice gives the same bits (rotation, mixed and full-sincos kernels)."""
    n = 5000 + 17
    res = []
    for block in (0, 32, 64, 128):
        ens = aw.Ensemble(n, tangent=tangent, wind=True, order=order)
        aw.aw_init_shell(ens, aw.make_grid(n, 1, -0.9, 0.9, angle_mode=1, lo_y=-0.3, hi_y=0.3), 1.0, 3e-2, 6)
        ens.block = block
        aw.aw_integrate(ens, n, 300, dt, 100)
        res.append(ens)
    for other in res[1:]:
        assert torch.equal(res[0].q, other.q) and torch.equal(res[0].acc, other.acc)
        assert torch.equal(res[0].wind, other.wind) and torch.equal(res[0].status, other.status)
        if tangent:
            assert torch.equal(res[0].w, other.w)
    bad = aw.Ensemble(64, tangent=False, wind=False)
    aw.aw_init_shell(bad, aw.make_grid(8, 8), 1.0, 1e-2, 0)
    bad.block = 96
    with pytest.raises(aw.AwError):
        aw.aw_integrate(bad, 64, 100, 0.01, 100)


@pytest.mark.parametrize("order,tangent,dt", [(4, True, 0.005), (4, True, 0.025), (6, True, 0.02), (6, False, 0.0628),
                                              (4, False, 0.1), (6, True, 0.15), (4, True, 0.2), (6, False, 1.0),
                                              (4, True, 1.2)])
def test_kernel_flavours_give_the_same_bits(aw, order, tangent, dt):
    """Every kernel exists in two ptxas schedules of the same source (throughput: source order for operand reuse;
    latency: interleaved chains for small ensembles); aw_integrate picks one from n.  Same arithmetic, same bits."""
    n = 3000 + 11
    res = []
    for flavour in (0, 1, 2):
        ens = aw.Ensemble(n, tangent=tangent, wind=True, order=order)
        aw.aw_init_shell(ens, aw.make_grid(n, 1, -0.9, 0.9, angle_mode=1, lo_y=-0.3, hi_y=0.3), 1.0, 3e-2, 6)
        ens.flavour = flavour
        aw.aw_integrate(ens, n, 400, dt, 100)
        res.append(ens)
    for other in res[1:]:
        assert torch.equal(res[0].q, other.q) and torch.equal(res[0].acc, other.acc)
        assert torch.equal(res[0].wind, other.wind) and torch.equal(res[0].status, other.status)
        if tangent:
            assert torch.equal(res[0].w, other.w)
    res[0].flavour = 3
    with pytest.raises(aw.AwError):
        aw.aw_integrate(res[0], n, 100, dt, 100)


# ------------------------------------------------------------------ odd histogram sizes, dropped points

def test_odd_histogram_sizes_with_dropped_points(aw, orc):
    """gx*gy odd: the 64-bit drop counter of aw_map_host's scratch sits at the next multiple of 8 bytes
    (AW_HIST_SCRATCH_BYTES), and aw_density refuses a misaligned counter instead of faulting."""
    cfg = aw.CONFIGS[3]
    gx, gy = 64, 32
    n = gx * gy
    a = aw.Ensemble(n, tangent=True, wind=True)
    aw.aw_init_shell(a, aw.make_grid(gx, gy, -1.0, 1.0, angle_mode=1), 1.0, cfg["eps"], 2)
    host_in = dict(q=a.q.cpu().pin_memory(), w=a.w.cpu().pin_memory(), acc=a.acc.cpu().pin_memory(),
                   wind=a.wind.cpu().pin_memory(), status=a.status[:n].cpu().pin_memory())
    for G, lo, hi in ((255, -0.5, 0.7), (1, -0.2, 0.2), (37, -1.0, 0.3)):
        b = aw.Ensemble(n, tangent=True, wind=True)
        b.c.E, b.c.eps = 1.0, cfg["eps"]
        scratch_bytes = (G * G * 4 + 7) // 8 * 8 + 8
        hist_dev = torch.empty(scratch_bytes // 4, dtype=torch.int32, device="cuda")
        out = dict(hist=torch.empty((G, G), dtype=torch.int32).pin_memory(),
                   dropped=torch.zeros(1, dtype=torch.int64).pin_memory(),
                   q=torch.empty((6, b.pitch), dtype=torch.float64).pin_memory(),
                   status=torch.empty(n, dtype=torch.uint8).pin_memory())
        aw.aw_map_host(b, host_in, 200, cfg["dt"], 100, aw.AW_IND_FLI, 0.0, (G, G), lo, hi, None, hist_dev, out)
        st = ensemble_to_oracle(b, orc)
        ref = np.zeros((G, G), dtype=np.uint32)
        d = orc.density(st, ref, lo, hi)
        assert int(d[0]) > 0                                     # points outside [lo, hi)^2 were dropped
        assert np.array_equal(out["hist"].numpy().view(np.uint32), ref) and out["dropped"].item() == int(d[0])
        assert int(ref.sum()) + int(d[0]) == int((st.status == 1).sum())
        # the device entry point with an odd histogram and its own aligned counter
        h2 = torch.zeros((G, G), dtype=torch.int32, device="cuda")
        d2 = torch.zeros(1, dtype=torch.int64, device="cuda")
        aw.aw_density(b, h2, lo, hi, 0, d2)
        assert np.array_equal(h2.cpu().numpy().view(np.uint32), ref) and d2.item() == int(d[0])
    # a counter at a 4-byte boundary is refused on the host
    h3 = torch.zeros(255 * 255 + 3, dtype=torch.int32, device="cuda")
    import ctypes as C
    from paper_1107_4107_b200.binding import lib
    rc = lib().aw_density(C.byref(b.c), C.c_void_p(h3.data_ptr()), 255, 255, -1.0, 1.0, 0,
                          C.c_void_p(h3.data_ptr() + 255 * 255 * 4))
    assert rc == -1
    torch.cuda.synchronize()                                     # and the context is still alive
    assert int(h3.sum().item()) == 0

"""Workload definitions (BASELINE.json configs[0..4]) as plain data.

No arithmetic of the method lives here: these are the parameters handed to aw_init_shell /
aw_integrate, shared by the tests (which pass the same numbers to the oracle) and by bench.py.
Inputs are synthetic and seeded: the paper's own initial conditions are random draws it does not print
(P:85); the configs take the shapes of its scans.
"""

# key: (grid, E, eps, seed, order, dt, steps, stride, tangent, outputs)
CONFIGS = {
    0: dict(name="cfg0_64x64_eps1e-2", gx=64, gy=64, lo=-1.0, hi=1.0, angle_mode=1, shape=0,
            cx=0.0, cy=0.0, r=0.0, E=1.0, eps=1e-2, seed=0, order=4, dt=0.01, steps=10_000,
            stride=100, tangent=False, density_every=0),
    1: dict(name="cfg1_512x512_eps1e-3_fli", gx=512, gy=512, lo=-1.0, hi=1.0, angle_mode=0, shape=0,
            cx=0.0, cy=0.0, r=0.0, E=1.0, eps=1e-3, seed=0, order=4, dt=0.01, steps=100_000,
            stride=100, tangent=True, density_every=0),
    2: dict(name="cfg2_1024x1024_eps1e-4_fli", gx=1024, gy=1024, lo=-1.0, hi=1.0, angle_mode=1, shape=0,
            cx=0.0, cy=0.0, r=0.0, E=1.0, eps=1e-4, seed=1, order=4, dt=0.02, steps=1_000_000,
            stride=100, tangent=True, density_every=0),
    3: dict(name="cfg3_2048x2048_eps3e-2_fli", gx=2048, gy=2048, lo=-1.0, hi=1.0, angle_mode=0, shape=0,
            cx=0.0, cy=0.0, r=0.0, E=1.0, eps=3e-2, seed=0, order=4, dt=0.005, steps=200_000,
            stride=100, tangent=True, density_every=0),
    4: dict(name="cfg4_diffusion_2^20", gx=1024, gy=1024, lo=-1.0, hi=1.0, angle_mode=1, shape=1,
            cx=0.0, cy=0.0, r=1e-3, E=1.0, eps=1e-3, seed=0, order=4, dt=0.01, steps=10_000_000,
            stride=100, tangent=False, density_every=10_000),
    # The paper's own workloads in its own units (eps = 1, T = 2 pi, h = 0.01 T, sixth-order scheme; P:55, P:85,
    # P:89): initial conditions uniform on the sphere S x torus, averaging window Dt = 50 T = 5000 steps, density of
    # the projected averaged velocity on the sphere (aw_mark + aw_density mode 3).  N = 2^22 stands in for the
    # paper's N ~ 1e8; the figures themselves cannot be compared (not in the container).
    5: dict(name="paper_fig2a_E400_sphere_velocity", gx=2048, gy=2048, lo=-1.0, hi=1.0, angle_mode=1, shape=3,
            cx=0.0, cy=0.0, r=0.0, E=400.0, eps=1.0, seed=2011, order=6, dt=0.06283185307179587, steps=5_000,
            stride=100, tangent=False, density_every=0, density_mode=3, hist_lo=-28.284271247461902,
            hist_hi=28.284271247461902),
    6: dict(name="paper_fig3a_E15_sphere_velocity", gx=2048, gy=2048, lo=-1.0, hi=1.0, angle_mode=1, shape=3,
            cx=0.0, cy=0.0, r=0.0, E=15.0, eps=1.0, seed=2011, order=6, dt=0.06283185307179587, steps=5_000,
            stride=100, tangent=False, density_every=0, density_mode=3, hist_lo=-5.477225575051661,
            hist_hi=5.477225575051661),
    # The paper's Fig. 4 workload: Gaussian cloud, sigma_vx = sigma_vy = 0.01, centred at the triple
    # resonance crossing W = (sqrt E, sqrt E, 0), uniform torus angles, v_z from the energy condition E = 15.  W lies
    # on the equator of S, so about half of the raw draws have 2(E - H_p(X)) < px^2 + py^2 and no real v_z: they are
    # drawn again (resample, R31) until on the shell, which gives the paper's N = 3.2e4 trajectories, all live.
    # eps = 1, sixth-order scheme, h = 0.01 T; the density of the projected averaged velocity is ACCUMULATED over
    # consecutive windows of Dt = 50 T ("averaged ... over the whole time span between consecutive plots"):
    # steps/window x (aw_mark; aw_integrate(Dt); aw_density mode 3).  The paper ran 2e5 such windows (t_p = 1e7 T,
    # 24 h on the Tesla M2050); the config times the first 20 (7) / 4 (8).  7: N = 3.2e4; 8: N = 2^20.
    7: dict(name="paper_fig4_E15_gauss_cloud_at_W", gx=200, gy=160, lo=-1.0, hi=1.0, angle_mode=1, shape=2,
            cx=3.872983346207417, cy=3.872983346207417, r=0.01, E=15.0, eps=1.0, seed=2011, order=6,
            dt=0.06283185307179587, steps=100_000, stride=100, tangent=False, density_every=0, density_mode=3,
            window=5_000, resample=40, hist_lo=-5.477225575051661, hist_hi=5.477225575051661),
    8: dict(name="paper_fig4_E15_gauss_cloud_at_W_2^20", gx=1024, gy=1024, lo=-1.0, hi=1.0, angle_mode=1, shape=2,
            cx=3.872983346207417, cy=3.872983346207417, r=0.01, E=15.0, eps=1.0, seed=2011, order=6,
            dt=0.06283185307179587, steps=20_000, stride=100, tangent=False, density_every=0, density_mode=3,
            window=5_000, resample=40, hist_lo=-5.477225575051661, hist_hi=5.477225575051661),
    # The paper's zooms (Figs. 2b,c / 3b,c): initial conditions uniformly distributed at random within a
    # small square segment of the sphere (seen along the third axis: a square in (px, py), R33), uniform torus angles,
    # v_z from the energy condition; "tracked only those trajectories which remained within the area during the whole
    # observation time" (survivor filter on the launch square, R25); averaging interval doubled to Dt = 100 T as for the
    # highest resolution (Fig. 3c); density of the projected averaged velocity over the same square.  The square
    # sits on the resonance plane px = py (Omega_(1,-1,0)) of the E = 15 shell; the paper does not print its own.
    9: dict(name="paper_fig3c_zoom_E15_square_survivors", gx=2048, gy=2048, lo=2.0, hi=2.5, angle_mode=1, shape=4,
            cx=0.0, cy=0.0, r=0.0, E=15.0, eps=1.0, seed=2011, order=6, dt=0.06283185307179587, steps=10_000,
            stride=100, tangent=False, density_every=0, density_mode=3, survive=True, hist_lo=2.0, hist_hi=2.5),
}

HIST_G = 1024          # density histogram is HIST_G x HIST_G over [HIST_LO, HIST_HI]^2 (configs[4])
HIST_LO, HIST_HI = -1.0, 1.0

# nominal fp64 flops per trajectory-step (FMA = 2, MUL/ADD = 1, sincos = 36)
NOMINAL_FLOPS = {(4, False): 384, (4, True): 498, (6, False): 896, (6, True): 1162}
# datasheet-derived fp64 FMA peak: 148 SMs x 64 DFMA/clk/SM x 2 flop x 1.965 GHz
FP64_PEAK_TFLOPS_NOMINAL = 148 * 64 * 2 * 1.965e9 / 1e12

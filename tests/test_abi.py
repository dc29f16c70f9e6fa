"""CPU-side checks of the boundary: libaw.so loads, exports every symbol include/aw.h declares, the
host helpers agree with the oracle's separately written ones, and argument validation happens on the
host before any launch (so it can be exercised without a GPU).  No compute calls here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def aw():
    from paper_1107_4107_b200 import build
    build.build()
    import paper_1107_4107_b200 as aw
    return aw


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "aw.h")).read()
    return sorted(set(re.findall(r"AW_API\s+[\w\s\*]+?\b(aw_\w+)\s*\(", src)))


def test_library_exports_every_declared_symbol(aw):
    names = declared_symbols()
    assert len(names) >= 16 and "aw_init_shell" in names and "aw_integrate" in names
    assert "aw_indicator" in names and "aw_density" in names
    L = C.CDLL(os.path.join(ROOT, "paper_1107_4107_b200", "libaw.so"))
    for n in names:
        assert hasattr(L, n), n
    assert aw.aw_version() == 210
    assert not any("probe" in n for n in names)            # probes live in tests/libaw_probe.so, not in the product ABI
    assert aw.aw_strerror(0) == "ok" and "invalid" in aw.aw_strerror(-1)


def test_probe_library_exports_its_header():
    """tests/aw_probe.h (test and measurement support) is a separate library built from the same device headers."""
    import aw_probe
    src = open(os.path.join(ROOT, "tests", "aw_probe.h")).read()
    names = sorted(set(re.findall(r"AWP_API\s+[\w\s\*]+?\b(awp_\w+)\s*\(", src)))
    assert names == ["awp_dfma_peak", "awp_dfma_shape", "awp_hamiltonian", "awp_sincos", "awp_tsincos", "awp_uniform"]
    L = C.CDLL(aw_probe.build())
    for n in names:
        assert hasattr(L, n), n
    assert L.awp_sincos(None, 4, None, None, None) == -1             # host-side validation, no device needed


def test_python_binding_has_the_same_names(aw):
    for n in declared_symbols():
        if n == "aw_last_cuda_error":
            continue
        assert hasattr(aw, n), n


def test_stage_constants_match_the_oracle(aw, orc):
    for order in (4, 6):
        for dt, eps in ((0.01, 1e-2), (-0.005, 3e-2), (0.02, 1e-4)):
            a, b = aw.aw_stage_constants(order, dt, eps)
            ao, bo = orc.stage_constants(order, dt, eps)
            assert len(a) == len(ao) and len(b) == len(bo)
            # order 4 is a closed form (bit-equal); order 6: library Newton (long double) vs the oracle's
            # mpmath literals -> both are the double nearest the same root
            assert np.allclose(a, ao, rtol=4e-16, atol=0) and np.allclose(b, bo, rtol=4e-16, atol=0)
            if order == 4:
                assert list(a) == list(ao) and list(b) == list(bo)
            assert abs(sum(a) - dt) < 4e-16 * abs(dt) * 8
    with pytest.raises(aw.AwError):
        aw.aw_stage_constants(5, 0.01, 1e-2)


def test_common_tangent_matches_the_oracle(aw, orc):
    for seed in (0, 1, 12345678901234567):
        t = np.array(aw.aw_common_tangent(seed))
        to = orc.common_tangent(seed)
        assert abs(np.linalg.norm(t) - 1) < 1e-15
        assert np.max(np.abs(t - to)) < 1e-15


def test_state_bytes(aw):
    b, pitch = aw.aw_state_bytes(4097, True, True)
    assert pitch == 4128 and b == 16 * pitch * 8 + 3 * pitch * 4 + 4097
    b, pitch = aw.aw_state_bytes(64, False, False)
    assert pitch == 64 and b == 10 * 64 * 8 + 64
    assert aw.aw_state_bytes(0)[1] == 0


def test_validation_happens_on_the_host(aw):
    """Bad arguments are rejected before any CUDA call: usable without a device."""
    from paper_1107_4107_b200.binding import AwState, Grid, lib
    L = lib()
    buf = (C.c_double * 1024)()
    base = C.addressof(buf)
    base += (-base) % 16
    st = AwState(64, 64, base, None, base, None, base, 1.0, 1e-2, 0.0, 0, 4, 1, 0, 0, None)
    g = Grid(8, 8, -1.0, 1.0, -1.0, 1.0, 0, 0, 0.0, 0.0, 0.0, 1, 0)
    EINVAL, ERANGE, ESTATE = -1, -3, -4
    assert L.aw_integrate(C.byref(st), 63, 100, 0.01, 100) == EINVAL        # n mismatch
    assert L.aw_integrate(C.byref(st), 64, 150, 0.01, 100) == EINVAL        # steps % stride
    assert L.aw_integrate(C.byref(st), 64, 100, 0.01, 0) == EINVAL          # stride <= 0
    assert L.aw_integrate(C.byref(st), 64, -100, 0.01, 100) == EINVAL       # steps < 0
    assert L.aw_integrate(C.byref(st), 64, 100, 0.0, 100) == EINVAL         # dt == 0
    assert L.aw_integrate(C.byref(st), 64, 100, float("nan"), 100) == EINVAL
    assert L.aw_integrate(C.byref(st), 64, 100000, 1.0, 100000) == ERANGE   # angle range (R7)
    assert L.aw_integrate(C.byref(st), 64, 0, 0.01, 100) == 0               # no-op
    st.order = 5
    assert L.aw_integrate(C.byref(st), 64, 100, 0.01, 100) == ESTATE
    st.order, st.ready = 4, 0
    assert L.aw_integrate(C.byref(st), 64, 100, 0.01, 100) == ESTATE
    st.ready = 1
    st.pitch = 70                                                          # not a multiple of 32
    assert L.aw_integrate(C.byref(st), 64, 100, 0.01, 100) == EINVAL
    st.pitch = 64
    st.q = base + 8                                                        # misaligned plane
    assert L.aw_integrate(C.byref(st), 64, 100, 0.01, 100) == EINVAL
    st.q = base
    # trigonometry level picked on the host from the largest drift angle (include/aw.h, aw_integrate)
    lv = lambda dt: L.aw_trig_level(C.byref(st), dt)
    assert [lv(0.005), lv(-0.005), lv(0.007), lv(0.01), lv(0.02), lv(0.03), lv(0.1), lv(0.15), lv(0.2), lv(0.5),
            lv(1.2)] == [1, 1, 2, 3, 4, 5, 6, 7, 8, 9, 0]
    st.order = 6                                      # largest |c_s| is 0.7845 instead of 1.3512
    assert [lv(0.005), lv(0.01), lv(0.02), lv(0.04), lv(0.05), lv(0.15), lv(0.3), lv(0.4), lv(1.0), lv(2.0)] == \
        [1, 2, 3, 4, 5, 6, 7, 8, 9, 0]
    st.order, st.trig = 4, 1
    assert lv(0.005) == 0
    st.trig = 0
    assert lv(0.0) == EINVAL
    # init_shell
    assert L.aw_init_shell(C.byref(st), C.byref(g), 1.0, 0.6, 0) == ERANGE  # E - 2|eps| <= 0
    g.gx = 7
    assert L.aw_init_shell(C.byref(st), C.byref(g), 1.0, 1e-2, 0) == EINVAL  # n > gx*gy: slice outside the ensemble
    g.gx, g.k0 = 8, 1
    assert L.aw_init_shell(C.byref(st), C.byref(g), 1.0, 1e-2, 0) == EINVAL  # k0 + n > gx*gy
    g.k0 = -1
    assert L.aw_init_shell(C.byref(st), C.byref(g), 1.0, 1e-2, 0) == EINVAL  # k0 < 0
    g.k0 = 0
    g.gx, g.hi_x = 8, -1.0
    assert L.aw_init_shell(C.byref(st), C.byref(g), 1.0, 1e-2, 0) == EINVAL  # hi <= lo
    g.hi_x, g.shape = 1.0, 7
    assert L.aw_init_shell(C.byref(st), C.byref(g), 1.0, 1e-2, 0) == EINVAL
    assert L.aw_init_shell(None, C.byref(g), 1.0, 1e-2, 0) == EINVAL
    # indicator / density
    assert L.aw_indicator(C.byref(st), 0, 0.0, base) == ESTATE              # FLI without tangent planes
    assert L.aw_indicator(C.byref(st), 9, 0.0, base) == EINVAL
    assert L.aw_indicator(C.byref(st), 2, 0.0, None) == EINVAL
    assert L.aw_density(C.byref(st), base, 16, 16, 1.0, -1.0, 0, None) == EINVAL
    assert L.aw_density(C.byref(st), base, 16, 16, -1.0, 1.0, 4, None) == EINVAL   # no such mode
    assert L.aw_density(C.byref(st), base, 16, 16, -1.0, 1.0, 1, None) == ESTATE   # velocity mode, no snapshot
    assert L.aw_indicator(C.byref(st), 4, 0.0, base) == ESTATE              # dP without a snapshot
    assert L.aw_mark(C.byref(st)) == ESTATE                                 # no qref planes
    st.qref = base
    st.tref, st.t = 0.0, 0.0
    assert L.aw_density(C.byref(st), base, 16, 16, -1.0, 1.0, 1, None) == ESTATE   # empty window t == tref
    assert L.aw_indicator(C.byref(st), 5, 0.0, base) == ESTATE
    # the averaged velocity needs the turn counters as well (a wrapped angle without its count would alias silently)
    st.t = 1.0
    assert st.wind is None
    assert L.aw_density(C.byref(st), base, 16, 16, -1.0, 1.0, 3, None) == ESTATE
    assert L.aw_indicator(C.byref(st), 6, 0.0, base) == ESTATE
    st.t, st.qref = 0.0, None
    # histogram / drop-counter alignment (uint32 / uint64 atomics)
    assert L.aw_density(C.byref(st), base + 2, 16, 16, -1.0, 1.0, 0, None) == EINVAL
    assert L.aw_density(C.byref(st), base, 16, 16, -1.0, 1.0, 0, base + 4) == EINVAL
    # block size: 0 (auto), 32, 64, 128
    st.block = 48
    assert L.aw_integrate(C.byref(st), 64, 100, 0.01, 100) == EINVAL
    st.block = 0
    st.flavour = 3                                                         # 0 auto, 1 throughput, 2 latency
    assert L.aw_integrate(C.byref(st), 64, 100, 0.01, 100) == EINVAL
    st.flavour = 0
    # aw_block_size: the smallest block whose grid is resident at once (16 blocks per SM; 6 for the trigonometry levels
    # that hold the 32 KB table in shared memory), 128 once that fills the chip (148 SMs assumed without a device)
    L.aw_block_size.argtypes = [C.POINTER(AwState), C.c_double]
    bs = AwState(); bs.E, bs.eps, bs.order = 1.0, 3e-2, 4
    def block(n, dt, order=4, E=1.0, eps=3e-2):
        bs.n, bs.order, bs.E, bs.eps = n, order, E, eps
        return L.aw_block_size(C.byref(bs), dt)
    assert [block(n, 0.005) for n in (1, 4096, 32000, 75648, 75649, 1 << 22)] == [32, 32, 32, 32, 128, 128]
    assert lv(0.005) == 1 and block(32000, 0.2) == 64            # level 8: table kernel, 1000 blocks of 32 > 148 x 6
    assert block(28000, 0.2) == 32 and block(57000, 0.2) == 128   # 875 blocks fit; 891 blocks of 64 do not
    assert block(32000, 0.0628, order=6, E=15.0, eps=1.0) == 64   # the paper's Fig. 4 ensemble
    # aw_kernel_schedule: latency flavour (0) up to 8 warps per sub-partition, throughput (1) beyond, where it exists
    L.aw_kernel_schedule.argtypes = [C.POINTER(AwState), C.c_double]
    def schedule(n, dt, flavour=0):
        bs.n, bs.order, bs.E, bs.eps, bs.flavour = n, 4, 1.0, 3e-2, flavour
        r = L.aw_kernel_schedule(C.byref(bs), dt)
        bs.flavour = 0
        return r
    assert [schedule(n, 0.005) for n in (4096, 151552, 151553, 1 << 22)] == [0, 0, 1, 1]
    assert schedule(1 << 22, 0.5) == 1 and schedule(4096, 1.2) == 0             # every level exists in both
    assert schedule(4096, 0.005, flavour=1) == 1 and schedule(1 << 22, 0.005, flavour=2) == 0
    assert schedule(4096, 0.005, flavour=3) == EINVAL
    bs.block = 128
    assert block(5, 0.005) == 128
    bs.block = 0
    assert block(5, 0.0) == EINVAL
    # Emax raises the energy bound the trig level (and the R7 range) is sized for; below E it is ignored
    st.Emax = 0.0
    assert lv(0.005) == 1
    st.Emax = 9.0
    assert lv(0.005) == 3 and L.aw_integrate(C.byref(st), 64, 300, 1.0, 300) == ERANGE
    st.Emax = float("nan")
    assert lv(0.005) == 1 and L.aw_integrate(C.byref(st), 64, 0, 1.0, 300) == 0
    st.Emax = 0.0
    assert L.aw_bound_energy(C.byref(st), None) == EINVAL
    assert L.aw_bound_energy(C.byref(st), base + 4) == EINVAL
    # aw_map_host / aw_velocity_map_host: everything is refused BEFORE the first copy is enqueued
    from paper_1107_4107_b200.binding import HostIn, HostOut
    hin = HostIn(base, None, base, None, base)
    hout = HostOut(base, base, None, None, None, None)
    mh = lambda *a: L.aw_map_host(C.byref(st), C.byref(hin), *a, C.byref(hout))
    assert mh(150, 0.01, 100, 2, 0.0, 16, 16, -1.0, 1.0, base, base) == EINVAL      # steps % stride
    assert mh(100, 0.01, 100, 12, 0.0, 16, 16, -1.0, 1.0, base, base) == EINVAL     # no such indicator kind
    assert mh(100, 0.01, 100, 0, 0.0, 16, 16, -1.0, 1.0, base, base) == ESTATE      # FLI without tangent planes
    assert mh(100, 0.01, 100, 5, 0.0, 16, 16, -1.0, 1.0, base, base) == ESTATE      # velocity kinds need a snapshot
    assert mh(100, 0.01, 100, 2, 0.0, 0, 16, -1.0, 1.0, base, base) == EINVAL       # gx <= 0
    assert mh(100, 0.01, 100, 2, 0.0, 16, 16, 1.0, -1.0, base, base) == EINVAL      # hi <= lo
    assert mh(100, 0.01, 100, 2, 0.0, 16, 16, -1.0, 1.0, None, base) == EINVAL      # image wanted, no scratch
    assert mh(100, 0.01, 100, 2, 0.0, 16, 16, -1.0, 1.0, base, base + 4) == EINVAL  # histogram scratch misaligned
    vm = lambda *a: L.aw_velocity_map_host(C.byref(st), C.byref(hin), *a, C.byref(hout))
    assert vm(100, 0.01, 100, 0, 16, 16, -1.0, 1.0, base) == EINVAL                 # mode 0 is not a velocity mode
    assert vm(100, 0.01, 100, 1, 16, 16, -1.0, 1.0, base) == ESTATE                 # no snapshot / counter planes
    assert vm(100, 0.01, 100, 1, 16, 0, -1.0, 1.0, base) == EINVAL
    # survivor filter: flag must be 0/1 and the rectangle non-empty
    st.survive = 2
    assert L.aw_integrate(C.byref(st), 64, 100, 0.01, 100) == EINVAL
    st.survive, st.surv_lo_x, st.surv_hi_x, st.surv_lo_y, st.surv_hi_y = 1, 0.5, 0.5, -1.0, 1.0
    assert L.aw_integrate(C.byref(st), 64, 100, 0.01, 100) == EINVAL
    st.survive = 0
    assert L.aw_density(C.byref(st), None, 16, 16, -1.0, 1.0, 0, None) == EINVAL
    assert L.aw_density(C.byref(st), base, 0, 16, -1.0, 1.0, 0, None) == EINVAL
    # zero-size ensemble: every call is a no-op that never reaches the device
    z = AwState(0, 0, None, None, None, None, None, 1.0, 1e-2, 0.0, 0, 4, 1, 0, 0, None)
    g0 = Grid(0, 0, -1.0, 1.0, -1.0, 1.0, 0, 0, 0.0, 0.0, 0.0, 1, 0)
    assert L.aw_integrate(C.byref(z), 0, 100, 0.01, 100) == 0
    assert L.aw_init_shell(C.byref(z), C.byref(g0), 1.0, 1e-2, 0) == EINVAL  # gx <= 0


def test_product_does_not_import_the_oracle():
    """The product path shares nothing with oracle/ (and has no CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_1107_4107_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "aw_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1107_4107_b200" not in src and "libaw.so" not in src, f

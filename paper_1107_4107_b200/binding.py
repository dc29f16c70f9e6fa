"""ctypes binding of libaw.so (include/aw.h).  Same names as the C entry points; marshalling only.

Tensors are torch CUDA tensors (device memory + stream come from PyTorch); every step of the path
runs inside the library's kernels.  If libaw.so is missing the import fails loudly — build it with
`python -m paper_1107_4107_b200.build` (or __graft_entry__.build()).
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libaw.so")

AW_OK, AW_EINVAL, AW_ECUDA, AW_ERANGE, AW_ESTATE = 0, -1, -2, -3, -4
AW_IND_FLI, AW_IND_FTLE, AW_IND_DH, AW_IND_CLASS = 0, 1, 2, 3
AW_IND_DP, AW_IND_VX, AW_IND_VY, AW_IND_VZ, AW_IND_DHS = 4, 5, 6, 7, 8
AW_DENS_ACTION, AW_DENS_VEL_UPPER, AW_DENS_VEL_LOWER, AW_DENS_VEL_BOTH = 0, 1, 2, 3
AW_SHAPE_GRID, AW_SHAPE_DISK, AW_SHAPE_GAUSS, AW_SHAPE_SPHERE, AW_SHAPE_RECT = 0, 1, 2, 3, 4
AW_ST_OFFSHELL, AW_ST_LIVE, AW_ST_NONFINITE, AW_ST_LEFT, AW_ST_RANGE = 0, 1, 2, 3, 4
AW_NOALLOC_MAX_N = 1 << 24      # aw_energy_stats_noalloc: size of the library's static scratch (include/aw.h)


class AwError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = lib().aw_strerror(code).decode()
        if code == AW_ECUDA:
            msg += " [cudaError %d]" % lib().aw_last_cuda_error()
        super().__init__("%s: %s (%d)" % (where, msg, code))


class AwState(C.Structure):
    _fields_ = [("n", C.c_int64), ("pitch", C.c_int64),
                ("q", C.c_void_p), ("w", C.c_void_p), ("acc", C.c_void_p), ("wind", C.c_void_p),
                ("status", C.c_void_p),
                ("E", C.c_double), ("eps", C.c_double), ("t", C.c_double), ("step", C.c_int64),
                ("order", C.c_int32), ("ready", C.c_int32), ("trig", C.c_int32), ("survive", C.c_int32),
                ("stream", C.c_void_p),
                ("qref", C.c_void_p), ("windref", C.c_void_p), ("tref", C.c_double),
                ("surv_lo_x", C.c_double), ("surv_hi_x", C.c_double),
                ("surv_lo_y", C.c_double), ("surv_hi_y", C.c_double),
                ("Emax", C.c_double), ("block", C.c_int32), ("flavour", C.c_int32)]


class Grid(C.Structure):
    _fields_ = [("gx", C.c_int32), ("gy", C.c_int32),
                ("lo_x", C.c_double), ("hi_x", C.c_double), ("lo_y", C.c_double), ("hi_y", C.c_double),
                ("angle_mode", C.c_int32), ("shape", C.c_int32),
                ("cx", C.c_double), ("cy", C.c_double), ("r", C.c_double),
                ("pz_sign", C.c_int32), ("tangent_mode", C.c_int32), ("k0", C.c_int64),
                ("resample", C.c_int32), ("reserved_", C.c_int32)]


class HostIn(C.Structure):
    _fields_ = [("q", C.c_void_p), ("w", C.c_void_p), ("acc", C.c_void_p), ("wind", C.c_void_p),
                ("status", C.c_void_p)]


class HostOut(C.Structure):
    _fields_ = [("image", C.c_void_p), ("hist", C.c_void_p), ("dropped", C.c_void_p),
                ("q", C.c_void_p), ("acc", C.c_void_p), ("status", C.c_void_p)]


def make_grid(gx, gy, lo=-1.0, hi=1.0, angle_mode=0, shape=0, cx=0.0, cy=0.0, r=0.0, pz_sign=1,
              tangent_mode=0, lo_y=None, hi_y=None, k0=0, resample=0):
    """The grid describes the WHOLE ensemble of gx*gy trajectories; an Ensemble of n trajectories initialised with
    it holds the slice [k0, k0 + n) (include/aw.h, aw_grid.k0)."""
    return Grid(gx, gy, lo, hi, lo if lo_y is None else lo_y, hi if hi_y is None else hi_y,
                angle_mode, shape, cx, cy, r, pz_sign, tangent_mode, k0, resample, 0)


_lib = None


def lib():
    """Load libaw.so (no silent fallback: a missing library is an error)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            raise ImportError("libaw.so not built: run `python -m paper_1107_4107_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(_LIBPATH)
        vp, i64, i32, dbl, u64 = C.c_void_p, C.c_int64, C.c_int32, C.c_double, C.c_uint64
        L.aw_strerror.restype = C.c_char_p
        L.aw_strerror.argtypes = [C.c_int]
        L.aw_last_cuda_error.restype = C.c_int
        L.aw_version.restype = C.c_int
        L.aw_launch_count.restype = u64
        L.aw_state_bytes.restype = C.c_size_t
        L.aw_state_bytes.argtypes = [i64, C.c_int, C.c_int, C.POINTER(i64)]
        L.aw_init_shell.argtypes = [C.POINTER(AwState), C.POINTER(Grid), dbl, dbl, u64]
        L.aw_integrate.argtypes = [C.POINTER(AwState), i64, i64, dbl, i64]
        L.aw_mark.argtypes = [C.POINTER(AwState)]
        L.aw_energy_stats_scratch_bytes.restype = C.c_size_t
        L.aw_energy_stats_scratch_bytes.argtypes = [i64]
        L.aw_energy_stats.argtypes = [C.POINTER(AwState), vp, vp]
        L.aw_energy_stats_noalloc.argtypes = [C.POINTER(AwState), vp]
        L.aw_indicator.argtypes = [C.POINTER(AwState), C.c_int, dbl, vp]
        L.aw_density.argtypes = [C.POINTER(AwState), vp, i32, i32, dbl, dbl, C.c_int, vp]
        L.aw_stage_constants.argtypes = [C.c_int, dbl, dbl, C.POINTER(dbl), C.POINTER(dbl)]
        L.aw_common_tangent.argtypes = [u64, C.POINTER(dbl)]
        L.aw_trig_level.argtypes = [C.POINTER(AwState), dbl]
        L.aw_map_host.argtypes = [C.POINTER(AwState), C.POINTER(HostIn), i64, dbl, i64, C.c_int, dbl,
                                  i32, i32, dbl, dbl, vp, vp, C.POINTER(HostOut)]
        L.aw_velocity_map_host.argtypes = [C.POINTER(AwState), C.POINTER(HostIn), i64, dbl, i64, C.c_int, i32, i32,
                                           dbl, dbl, vp, C.POINTER(HostOut)]
        L.aw_bound_energy.argtypes = [C.POINTER(AwState), vp]
        L.aw_block_size.argtypes = [C.POINTER(AwState), dbl]
        L.aw_kernel_schedule.argtypes = [C.POINTER(AwState), dbl]
        _lib = L
    return _lib


def _check(rc, where):
    if rc < 0:
        raise AwError(rc, where)
    return rc


def _stream_ptr(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


# ------------------------------------------------------------------------------ host helpers

def aw_version():
    return lib().aw_version()


def aw_strerror(code):
    return lib().aw_strerror(code).decode()


def aw_launch_count():
    return int(lib().aw_launch_count())


def aw_state_bytes(n, with_tangent=True, with_wind=True):
    pitch = C.c_int64(0)
    b = lib().aw_state_bytes(n, int(with_tangent), int(with_wind), C.byref(pitch))
    return int(b), int(pitch.value)


def aw_stage_constants(order, dt, eps):
    a = (C.c_double * 8)()
    b = (C.c_double * 7)()
    S = _check(lib().aw_stage_constants(order, dt, eps, a, b), "aw_stage_constants")
    return list(a[:S + 1]), list(b[:S])


def aw_trig_level(ens, dt):
    return _check(lib().aw_trig_level(C.byref(ens.c), dt), "aw_trig_level")


def aw_block_size(ens, dt):
    return _check(lib().aw_block_size(C.byref(ens.c), dt), "aw_block_size")


def aw_kernel_schedule(ens, dt):
    return _check(lib().aw_kernel_schedule(C.byref(ens.c), dt), "aw_kernel_schedule")


def aw_common_tangent(seed):
    t = (C.c_double * 6)()
    _check(lib().aw_common_tangent(seed, t), "aw_common_tangent")
    return list(t)


# ------------------------------------------------------------------------------ ensemble state

class Ensemble:
    """Caller-owned SoA planes (torch CUDA tensors) + the aw_state struct that points at them."""

    def __init__(self, n, tangent=True, wind=True, order=4, device="cuda:0", ref=False):
        _, pitch = aw_state_bytes(n, tangent, wind)
        self.n, self.pitch = int(n), pitch
        dev = torch.device(device)
        self.device = dev
        self.q = torch.zeros((6, pitch), dtype=torch.float64, device=dev)
        self.w = torch.zeros((6, pitch), dtype=torch.float64, device=dev) if tangent else None
        self.acc = torch.zeros((4, pitch), dtype=torch.float64, device=dev)
        self.wind = torch.zeros((3, pitch), dtype=torch.int32, device=dev) if wind else None
        self.status = torch.zeros((max(n, 1),), dtype=torch.uint8, device=dev)
        self.c = AwState(n, pitch, self.q.data_ptr(), self.w.data_ptr() if tangent else None,
                         self.acc.data_ptr(), self.wind.data_ptr() if wind else None,
                         self.status.data_ptr(), float("nan"), float("nan"), 0.0, 0, order, 0, 0, 0, None)
        # snapshot planes for aw_mark (window start of P:67 / P(0) of P:37); allocated on request
        self.qref = torch.zeros((6, pitch), dtype=torch.float64, device=dev) if ref else None
        self.windref = torch.zeros((3, pitch), dtype=torch.int32, device=dev) if (ref and wind) else None
        if ref:
            self.c.qref = self.qref.data_ptr()
            self.c.windref = self.windref.data_ptr() if wind else None

    # plain-data views of the struct
    E = property(lambda s: s.c.E)
    eps = property(lambda s: s.c.eps)
    t = property(lambda s: s.c.t)
    step = property(lambda s: s.c.step)
    tref = property(lambda s: s.c.tref)
    Emax = property(lambda s: s.c.Emax)

    def set_survivors(self, rect):
        """rect = (lo_x, hi_x, lo_y, hi_y) switches the survivor filter of P:99 on; None switches it off."""
        if rect is None:
            self.c.survive = 0
        else:
            self.c.survive = 1
            self.c.surv_lo_x, self.c.surv_hi_x, self.c.surv_lo_y, self.c.surv_hi_y = rect

    @property
    def order(self):
        return self.c.order

    @order.setter
    def order(self, v):
        self.c.order = v

    @property
    def block(self):
        return self.c.block

    @block.setter
    def block(self, v):
        self.c.block = v

    @property
    def flavour(self):
        return self.c.flavour

    @flavour.setter
    def flavour(self, v):
        self.c.flavour = v

    @property
    def trig(self):
        return self.c.trig

    @trig.setter
    def trig(self, v):
        self.c.trig = v

    def bind_stream(self, stream=None):
        self.c.stream = _stream_ptr(stream)

    def load_host(self, q, w, acc, wind, status, E, eps, t=0.0, step=0):
        """Upload a host state (numpy arrays shaped like the planes) and mark the struct ready."""
        self.q.copy_(torch.from_numpy(q))
        if self.w is not None:
            self.w.copy_(torch.from_numpy(w))
        self.acc.copy_(torch.from_numpy(acc))
        if self.wind is not None and wind is not None:
            self.wind.copy_(torch.from_numpy(wind))
        self.status[:self.n].copy_(torch.from_numpy(status))
        self.c.E, self.c.Emax, self.c.eps, self.c.t, self.c.step, self.c.ready = E, E, eps, t, step, 1


def aw_init_shell(ens, grid, E, eps, seed, stream=None):
    ens.bind_stream(stream)
    _check(lib().aw_init_shell(C.byref(ens.c), C.byref(grid), E, eps, seed), "aw_init_shell")
    return ens


def aw_integrate(ens, n, steps, dt, stride, stream=None):
    ens.bind_stream(stream)
    _check(lib().aw_integrate(C.byref(ens.c), n, steps, dt, stride), "aw_integrate")
    return ens


def aw_bound_energy(ens, stream=None):
    """Synchronous: ens.Emax <- max over live trajectories of H(X,P), from the data (include/aw.h)."""
    ens.bind_stream(stream)
    scratch = torch.zeros((1,), dtype=torch.int64, device=ens.device)
    _check(lib().aw_bound_energy(C.byref(ens.c), _ptr(scratch)), "aw_bound_energy")
    return ens.c.Emax


def aw_mark(ens, stream=None):
    ens.bind_stream(stream)
    _check(lib().aw_mark(C.byref(ens.c)), "aw_mark")
    return ens


def aw_indicator(ens, kind, thr=0.0, out=None, stream=None):
    ens.bind_stream(stream)
    if out is None:
        out = torch.empty((max(ens.n, 1),), dtype=torch.uint8 if kind == AW_IND_CLASS else torch.float64,
                          device=ens.device)
    _check(lib().aw_indicator(C.byref(ens.c), kind, thr, _ptr(out)), "aw_indicator")
    return out[:ens.n]


def aw_energy_stats_scratch_bytes(n):
    return int(lib().aw_energy_stats_scratch_bytes(n))


def aw_energy_stats(ens, out=None, stream=None):
    """8 doubles on the device: live count, max / mean / rms of dH_max, mean / rms of the signed final error,
    index of the worst trajectory, max |signed error| (include/aw.h)."""
    ens.bind_stream(stream)
    scratch = torch.empty((aw_energy_stats_scratch_bytes(ens.n) + 7) // 8, dtype=torch.float64, device=ens.device)
    if out is None:
        out = torch.empty((8,), dtype=torch.float64, device=ens.device)
    _check(lib().aw_energy_stats(C.byref(ens.c), _ptr(scratch), _ptr(out)), "aw_energy_stats")
    return out


def aw_energy_stats_noalloc(ens, out, stream=None):
    """aw_energy_stats without any allocation: the scratch is a static device array inside libaw.so (at most
    AW_NOALLOC_MAX_N trajectories); `out` is the caller's 8-double CUDA tensor.  Calls that overlap on the GPU race
    on the shared scratch (include/aw.h)."""
    ens.bind_stream(stream)
    _check(lib().aw_energy_stats_noalloc(C.byref(ens.c), _ptr(out)), "aw_energy_stats_noalloc")
    return out


def aw_density(ens, hist, lo, hi, mode=0, dropped=None, stream=None):
    """hist: uint32-as-int32 CUDA tensor [gy, gx] (torch has no uint32 arithmetic; the bits are uint32).
    dropped: int64 CUDA tensor [1] or None.  ADDS into hist."""
    ens.bind_stream(stream)
    gy, gx = hist.shape
    _check(lib().aw_density(C.byref(ens.c), _ptr(hist), gx, gy, lo, hi, mode, _ptr(dropped)), "aw_density")
    return hist


def aw_map_host(ens, host_in, steps, dt, stride, kind, thr, hist_shape, lo, hi, ind_dev, hist_dev,
                host_out, stream=None):
    """host_in / host_out: dicts of pinned (or pageable) CPU torch tensors; see include/aw.h."""
    ens.bind_stream(stream)
    hin = HostIn(_ptr(host_in["q"]), _ptr(host_in.get("w")), _ptr(host_in["acc"]),
                 _ptr(host_in.get("wind")), _ptr(host_in["status"]))
    hout = HostOut(_ptr(host_out.get("image")), _ptr(host_out.get("hist")), _ptr(host_out.get("dropped")),
                   _ptr(host_out.get("q")), _ptr(host_out.get("acc")), _ptr(host_out.get("status")))
    gy, gx = hist_shape
    _check(lib().aw_map_host(C.byref(ens.c), C.byref(hin), steps, dt, stride, kind, thr, gx, gy, lo, hi,
                             _ptr(ind_dev), _ptr(hist_dev), C.byref(hout)), "aw_map_host")


def aw_velocity_map_host(ens, host_in, steps, dt, stride, mode, hist_shape, lo, hi, hist_dev, host_out, stream=None):
    """The paper's pipeline with host buffers: upload, aw_mark, aw_integrate, aw_density(mode 1..3), download."""
    ens.bind_stream(stream)
    hin = HostIn(_ptr(host_in["q"]), _ptr(host_in.get("w")), _ptr(host_in["acc"]),
                 _ptr(host_in.get("wind")), _ptr(host_in["status"]))
    hout = HostOut(None, _ptr(host_out.get("hist")), _ptr(host_out.get("dropped")),
                   _ptr(host_out.get("q")), _ptr(host_out.get("acc")), _ptr(host_out.get("status")))
    gy, gx = hist_shape
    _check(lib().aw_velocity_map_host(C.byref(ens.c), C.byref(hin), steps, dt, stride, mode, gx, gy, lo, hi,
                                      _ptr(hist_dev), C.byref(hout)), "aw_velocity_map_host")

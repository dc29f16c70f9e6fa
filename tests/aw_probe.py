"""ctypes loader of tests/libaw_probe.so (tests/aw_probe.h): TEST AND MEASUREMENT SUPPORT, not the product.

The probes compile the library's own device headers (csrc/aw_trig.cuh, aw_model.cuh, aw_internal.cuh) into small
elementwise kernels so that the tests can check the integrator's sincos, the counter-based generator and the
Hamiltonian routine in isolation; bench.py uses the two DFMA micro-benchmarks to print a measured fp64 peak beside
the derived one.  `python tests/aw_probe.py` builds the library (nvcc, sm_100a; cross-compiles without a GPU).
"""
import ctypes as C
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "aw_probe.cu")
_LIB = os.path.join(_HERE, "libaw_probe.so")
_CSRC = os.path.join(os.path.dirname(_HERE), "paper_1107_4107_b200", "csrc")
_DEPS = [_SRC, os.path.join(_HERE, "aw_probe.h")] + [os.path.join(_CSRC, f) for f in
                                                    ("aw_internal.cuh", "aw_trig.cuh", "aw_trig_coeffs.h", "aw_model.cuh",
                                                     "aw_tsincos.cuh", "aw_trig_table.h")]
_lib = None


def build(force=False):
    if not force and os.path.exists(_LIB) and all(os.path.getmtime(d) <= os.path.getmtime(_LIB) for d in _DEPS):
        return _LIB
    nvcc = os.environ.get("NVCC") or ("/usr/local/cuda/bin/nvcc" if os.path.exists("/usr/local/cuda/bin/nvcc") else "nvcc")
    tmp = _LIB + ".%d.tmp" % os.getpid()
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
           "-Xcompiler", "-fvisibility=hidden", "-shared", "-o", tmp, _SRC, "-lcudart"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed on tests/aw_probe.cu")
    os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, i64, dbl, u64 = C.c_void_p, C.c_int64, C.c_double, C.c_uint64
        L.awp_sincos.argtypes = [vp, i64, vp, vp, vp]
        L.awp_tsincos.argtypes = [vp, i64, vp, vp, vp]
        L.awp_uniform.argtypes = [u64, u64, i64, C.c_uint32, vp, vp]
        L.awp_hamiltonian.argtypes = [vp, i64, i64, dbl, vp, vp]
        L.awp_dfma_peak.argtypes = [C.c_int, C.c_int, C.c_int, i64, vp, C.POINTER(dbl), C.POINTER(dbl), vp]
        L.awp_dfma_shape.argtypes = [C.c_int, C.c_int, C.c_int, i64, vp, C.POINTER(dbl), C.POINTER(dbl), vp]
        _lib = L
    return _lib


def _ok(rc, where):
    if rc != 0:
        raise RuntimeError("%s failed (%d)" % (where, rc))


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def sincos(x):
    import torch
    s, c = torch.empty_like(x), torch.empty_like(x)
    _ok(lib().awp_sincos(C.c_void_p(x.data_ptr()), x.numel(), C.c_void_p(s.data_ptr()), C.c_void_p(c.data_ptr()),
                         _stream()), "awp_sincos")
    return s, c


def tsincos(x):
    """The table-driven sincos of the integrator's step loop (csrc/aw_tsincos.cuh)."""
    import torch
    s, c = torch.empty_like(x), torch.empty_like(x)
    _ok(lib().awp_tsincos(C.c_void_p(x.data_ptr()), x.numel(), C.c_void_p(s.data_ptr()), C.c_void_p(c.data_ptr()),
                          _stream()), "awp_tsincos")
    return s, c


def uniform(seed, k0, n, slot, device="cuda:0"):
    import torch
    out = torch.empty((n,), dtype=torch.float64, device=device)
    _ok(lib().awp_uniform(seed, k0, n, slot, C.c_void_p(out.data_ptr()), _stream()), "awp_uniform")
    return out


def hamiltonian(q, n, pitch, eps):
    import torch
    out = torch.empty((n,), dtype=torch.float64, device=q.device)
    _ok(lib().awp_hamiltonian(C.c_void_p(q.data_ptr()), n, pitch, eps, C.c_void_p(out.data_ptr()), _stream()),
        "awp_hamiltonian")
    return out


def dfma_peak(blocks, threads, chains, iters, device="cuda:0"):
    """(milliseconds, DFMA thread-instructions)"""
    import torch
    sink = torch.zeros((2,), dtype=torch.float64, device=device)
    ms, cnt = C.c_double(0), C.c_double(0)
    _ok(lib().awp_dfma_peak(blocks, threads, chains, iters, C.c_void_p(sink.data_ptr()), C.byref(ms), C.byref(cnt),
                            _stream()), "awp_dfma_peak")
    return ms.value, cnt.value


def dfma_shape(blocks, threads, shape, iters, device="cuda:0"):
    """(milliseconds, fp64 thread-instructions) for one operand shape (tests/aw_probe.h)"""
    import torch
    work = torch.zeros((160,), dtype=torch.float64, device=device)
    ms, cnt = C.c_double(0), C.c_double(0)
    _ok(lib().awp_dfma_shape(blocks, threads, shape, iters, C.c_void_p(work.data_ptr()), C.byref(ms), C.byref(cnt),
                             _stream()), "awp_dfma_shape")
    return ms.value, cnt.value


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))

"""Build libaw.so (the C-ABI CUDA library, include/aw.h) in-tree with nvcc for sm_100a.

    python -m paper_1107_4107_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU; the .so is git-ignored but travels to the GPU box with gpurun.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libaw.so")
SOURCES = ["aw_api.cu", "aw_integrate.cu", "aw_init.cu", "aw_reduce.cu"]
# (source, object, extra flags): aw_integrate.cu is compiled a second time for the rotation kernels (trig levels 1-7) with
# ptxas -O1, whose scheduling keeps operand-sharing FMAs adjacent (see the comment at AW_LEVEL_GROUP in the source)
UNITS = [("aw_api.cu", "aw_api.o", []), ("aw_integrate.cu", "aw_integrate.o", []),
         ("aw_integrate.cu", "aw_integrate_low.o", ["-DAW_LEVEL_GROUP=1", "-Xptxas", "-O1"]),
         ("aw_init.cu", "aw_init.o", []), ("aw_reduce.cu", "aw_reduce.o", [])]
HEADERS = ["aw_internal.cuh", "aw_trig.cuh", "aw_trig_coeffs.h", "aw_trig_table.h", "aw_tsincos.cuh", "aw_model.cuh", os.path.join("..", "..", "include", "aw.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "-Xptxas", "-v"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def source_hash():
    """16 hex digits identifying what libaw.so is built from: every source and header with comments and blank
    space removed (an edit that changes no code keeps the hash) and the compiler flags.  bench.py quotes an
    ncu-measured DRAM traffic figure only when it was captured on the same build (profiles/traffic_by_build.csv)."""
    import hashlib
    import re
    h = hashlib.sha256()
    for f in sorted(set(SOURCES + HEADERS)):
        text = open(os.path.join(CSRC, f), encoding="utf-8").read()
        text = re.sub(r"/\*.*?\*/", " ", text, flags=re.S)        # block comments
        text = re.sub(r"//[^\n]*", " ", text)                     # line comments (no string literal here holds //)
        h.update(f.encode())
        h.update(" ".join(text.split()).encode())
    h.update(repr((NVCC_FLAGS, UNITS)).encode())
    return h.hexdigest()[:16]


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False, extra_flags=()):
    """Compile csrc/*.cu -> paper_1107_4107_b200/libaw.so.  Returns the path."""
    if not force and not needs_build():
        return LIB
    objs = []
    build_dir = os.path.join(HERE, "build")
    os.makedirs(build_dir, exist_ok=True)
    log = []
    extra_flags = list(extra_flags) + os.environ.get("AW_EXTRA_NVCC_FLAGS", "").split()   # tuning experiments only
    for src, objname, unit_flags in UNITS:
        obj = os.path.join(build_dir, objname)
        cmd = [_nvcc()] + NVCC_FLAGS + unit_flags + extra_flags + ["-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        log.append(r.stderr)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("nvcc failed on " + src)
        objs.append(obj)
    tmp = LIB + ".%d.tmp" % os.getpid()
    cmd = [_nvcc(), "-shared", "-o", tmp] + objs + ["-lcudart"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("link failed")
    os.replace(tmp, LIB)
    with open(os.path.join(build_dir, "ptxas.log"), "w") as f:
        f.write("\n".join(log))
    if verbose:
        sys.stderr.write("\n".join(log))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))

"""aw_energy_stats_noalloc (include/aw.h): the energy-drift statistics with the block partials in a static device
array inside libaw.so instead of caller-provided scratch, for callers that cannot allocate device memory.  It runs
the same two kernels as aw_energy_stats, so the bar is the one test_energy_drift_statistics_parity sets for two runs
of that reduction: identical bits.  Two calls in a row on DIFFERENT ensembles (the second one smaller, so that a
partial left over from the first call would be folded in if the entry point read beyond what it wrote), then the
first ensemble again; no device memory is allocated inside the calls; sizes beyond AW_NOALLOC_MAX_N are refused.

Collected last on purpose (pytest -x: a failure here hides nothing after it).  Passes alone in a
fresh process (the first call does the per-device address look-up) and after the other tests.
"""
import numpy as np
import pytest
import torch

gpu = pytest.mark.gpu


def test_library_imports_no_allocating_cuda_routine():
    """No GPU needed: libaw.so links the CUDA runtime dynamically, so its import table lists every runtime call it
    can make.  No cudaMalloc* / cudaFree* / cudaHostAlloc / memory-pool routine is among them (the library never
    allocates: every buffer is the caller's, include/aw.h), and cudaGetSymbolAddress — the static scratch's address
    look-up — is."""
    import subprocess
    from paper_1107_4107_b200 import build
    names = [l.split()[-1].split("@")[0] for l in
             subprocess.run(["nm", "-D", "--undefined-only", build.build()], capture_output=True, text=True,
                            check=True).stdout.splitlines() if l.strip()]
    cuda = [n for n in names if n.startswith("cuda") or n.startswith("cu") and n[2:3].isupper()]
    assert "cudaGetSymbolAddress" in cuda and "cudaLaunchKernel" in cuda
    bad = [n for n in cuda if any(w in n for w in ("Malloc", "Free", "Alloc", "MemPool", "Create", "Destroy"))]
    assert not bad, bad


@pytest.fixture(scope="module")
def aw():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1107_4107_b200 import build
    build.build()
    import paper_1107_4107_b200 as aw
    return aw


def _ensemble(aw, gx, gy, seed, steps):
    n = gx * gy
    ens = aw.Ensemble(n, tangent=False, wind=True)
    aw.aw_init_shell(ens, aw.make_grid(gx, gy, -1.02, 1.02, angle_mode=1), 1.0, 1e-2, seed)   # corners off the shell
    aw.aw_integrate(ens, n, steps, 0.02, 100)
    return ens


@gpu
def test_noalloc_energy_stats_equals_the_caller_scratch_path_twice_in_a_row(aw):
    big = _ensemble(aw, 521, 301, 5, 300)          # 156 821 trajectories: 77 block partials, ragged tail
    small = _ensemble(aw, 67, 33, 6, 500)          # 2 211 trajectories: 2 block partials
    want_big = aw.aw_energy_stats(big).cpu().numpy()
    want_small = aw.aw_energy_stats(small).cpu().numpy()
    assert want_big[0] > 100_000 and 0 < want_small[0] <= 2211 and want_big[1] > 0 and want_small[1] > 0
    assert not np.array_equal(want_big, want_small)

    out = torch.full((3, 8), -1.0, dtype=torch.float64, device="cuda")     # caller-owned outputs
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated(), torch.cuda.memory_reserved()
    free_before, _ = torch.cuda.mem_get_info()
    aw.aw_energy_stats_noalloc(big, out[0])
    aw.aw_energy_stats_noalloc(small, out[1])      # straight after, same stream: must not see the 75 stale partials
    aw.aw_energy_stats_noalloc(big, out[2])
    torch.cuda.synchronize()
    assert (torch.cuda.memory_allocated(), torch.cuda.memory_reserved()) == before
    got = out.cpu().numpy()
    assert np.array_equal(got[0], want_big, equal_nan=True)
    assert np.array_equal(got[1], want_small, equal_nan=True)
    assert np.array_equal(got[2], want_big, equal_nan=True)
    # once the per-device look-up is done (first call above), further calls leave the device's free memory alone
    free_mid, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        aw.aw_energy_stats_noalloc(small, out[1])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_mid and free_mid <= free_before
    assert np.array_equal(out[1].cpu().numpy(), want_small, equal_nan=True)


@gpu
def test_noalloc_energy_stats_empty_and_all_masked(aw):
    out = torch.full((8,), -1.0, dtype=torch.float64, device="cuda")
    ens = _ensemble(aw, 67, 33, 6, 100)
    ens.status.zero_()                              # nobody live: count 0, NaN means, index -1 — and nothing stale
    aw.aw_energy_stats_noalloc(ens, out)
    assert np.array_equal(out.cpu().numpy(), aw.aw_energy_stats(ens).cpu().numpy(), equal_nan=True)
    assert out[0].item() == 0.0 and out[6].item() == -1.0 and np.isnan(out[2].item())
    empty = aw.Ensemble(0, tangent=False, wind=False)
    empty.c.E, empty.c.eps, empty.c.ready = 1.0, 1e-2, 1
    aw.aw_energy_stats_noalloc(empty, out)
    assert np.array_equal(out.cpu().numpy(), aw.aw_energy_stats(empty).cpu().numpy(), equal_nan=True)
    assert out[0].item() == 0.0


@gpu
def test_noalloc_energy_stats_refuses_sizes_beyond_its_scratch(aw):
    """Validation happens on the host before anything is launched, so the struct may describe more trajectories than
    its planes hold: the call must return AW_ERANGE without touching them."""
    assert aw.AW_NOALLOC_MAX_N == 1 << 24
    ens = _ensemble(aw, 67, 33, 6, 100)
    out = torch.full((8,), -1.0, dtype=torch.float64, device="cuda")
    launches = aw.aw_launch_count()
    n, pitch = ens.c.n, ens.c.pitch
    try:
        ens.c.n, ens.c.pitch = aw.AW_NOALLOC_MAX_N + 1, aw.AW_NOALLOC_MAX_N + 32
        with pytest.raises(aw.AwError) as e:
            aw.aw_energy_stats_noalloc(ens, out)
        assert e.value.code == -3 and "range" in str(e.value)            # AW_ERANGE
    finally:
        ens.c.n, ens.c.pitch = n, pitch
    assert aw.aw_launch_count() == launches
    torch.cuda.synchronize()
    assert torch.all(out == -1.0)
    with pytest.raises(aw.AwError) as e:                                 # the other errors are aw_energy_stats's
        aw.aw_energy_stats_noalloc(ens, None)
    assert e.value.code == -1
    odd = torch.zeros((9,), dtype=torch.float64, device="cuda")[1:]      # 8 doubles, 8 bytes off a 16-byte boundary
    with pytest.raises(aw.AwError) as e:
        aw.aw_energy_stats_noalloc(ens, odd)
    assert e.value.code == -1                                            # out_dev not 16-byte aligned
    aw.aw_energy_stats_noalloc(ens, out)                                 # and the state is still usable
    assert np.array_equal(out.cpu().numpy(), aw.aw_energy_stats(ens).cpu().numpy(), equal_nan=True)

"""Two ranks, ONE GPU, gloo: the sharded job with the real CUDA kernels as per-rank compute equals the single-process
GPU result bit for bit (image) and count for count (histogram), in both scaling modes, for the grid with seeded
angles and for a cloud.  The ranks never wait on one another inside a kernel (the only exchanges are the histogram
all-reduce and the image gather between kernels, done here on host copies because NCCL needs one device per rank and
this box has one).  Timing of N > 1 is not measured anywhere in this repository (no multi-GPU hardware in this run)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu

CASES = {
    # name: (gx, gy, shape, angle_mode, cx, cy, r, E, eps, order, dt)
    "grid_seeded": (64, 30, 0, 1, 0.0, 0.0, 0.0, 1.0, 3e-2, 4, 0.005),
    "gauss_cloud_at_W": (64, 25, 2, 1, 15.0 ** 0.5, 15.0 ** 0.5, 0.01, 15.0, 1.0, 6, 0.0628),
}


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _run(gx, gy_total, k0, n, case, steps):
    import paper_1107_4107_b200 as aw
    _, _, shape, angle_mode, cx, cy, r, E, eps, order, dt = CASES[case]
    ens = aw.Ensemble(n, tangent=True, wind=True, order=order)
    g = aw.make_grid(gx, gy_total, -1.0, 1.0, angle_mode, shape, cx, cy, r, k0=k0, resample=20 if shape == 2 else 0)
    aw.aw_init_shell(ens, g, E, eps, 3)
    aw.aw_integrate(ens, n, steps, dt, 100)
    fli = aw.aw_indicator(ens, aw.AW_IND_FLI)
    hist = torch.zeros((64, 64), dtype=torch.int32, device="cuda")
    lim = 1.1 * (2 * E) ** 0.5
    aw.aw_density(ens, hist, -lim, lim)
    torch.cuda.synchronize()
    return fli.cpu(), hist.cpu()


def _worker(rank, world, port, case, scaling, steps, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    from paper_1107_4107_b200 import parallel
    gx, gy = CASES[case][:2]
    gxt, gyt, k0, n = parallel.slice_of(gx, gy, world, rank, scaling)
    fli, hist = _run(gxt, gyt, k0, n, case, steps)
    parallel.allreduce_hist(hist)
    counts = [parallel.slice_of(gx, gy, world, rr, scaling)[3] for rr in range(world)]
    img = parallel.gather_image(fli, counts)
    if rank == 0:
        np.save(os.path.join(out_dir, "img.npy"), img.numpy())
        np.save(os.path.join(out_dir, "hist.npy"), hist.numpy())
    dist.destroy_process_group()


@pytest.mark.parametrize("case,scaling", [("grid_seeded", "strong"), ("grid_seeded", "weak"), ("gauss_cloud_at_W", "weak")])
def test_two_ranks_on_one_gpu_equal_the_single_process_result(tmp_path, case, scaling):
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1107_4107_b200 import build
    build.build()
    world, steps = 2, 300
    mp.spawn(_worker, args=(world, _free_port(), case, scaling, steps, str(tmp_path)), nprocs=world, join=True)
    gx, gy = CASES[case][:2]
    gy_total = gy * world if scaling == "weak" else gy
    ref_img, ref_hist = _run(gx, gy_total, 0, gx * gy_total, case, steps)
    img, hist = np.load(tmp_path / "img.npy"), np.load(tmp_path / "hist.npy")
    assert np.array_equal(img, ref_img.numpy(), equal_nan=True)
    assert np.array_equal(hist, ref_hist.numpy()) and hist.sum() > 0


def _nccl_worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", 0))
    from paper_1107_4107_b200 import parallel
    parallel._active = lambda: True                        # a world of one still goes through the collectives
    hist = torch.arange(-8, 8, dtype=torch.int32, device="cuda").reshape(4, 4).contiguous()
    before = hist.clone()
    parallel.allreduce_hist(hist)
    img = parallel.gather_image(torch.arange(5, dtype=torch.float64, device="cuda"), [5])
    ok = torch.equal(hist, before) and img.is_cuda and torch.equal(img.cpu(), torch.arange(5, dtype=torch.float64))
    cls = parallel.gather_image(torch.arange(7, dtype=torch.uint8, device="cuda"), [7])     # CLASS images are bytes
    ok = ok and torch.equal(cls.cpu(), torch.arange(7, dtype=torch.uint8))
    open(os.path.join(out_dir, "ok"), "w").write(str(bool(ok)))
    dist.destroy_process_group()


def test_nccl_collectives_on_device_tensors(tmp_path):
    """bench.py's N > 1 path calls NCCL all_reduce on the int32 histogram and NCCL gather on the fp64 (or uint8) image
    where they live, on the device.  With one GPU the communicator has one rank; this checks that the calls are the
    ones NCCL accepts for these dtypes and shapes (the exchange itself is trivial)."""
    assert torch.cuda.is_available()
    mp.spawn(_nccl_worker, args=(1, _free_port(), str(tmp_path)), nprocs=1, join=True)
    assert open(tmp_path / "ok").read() == "True"

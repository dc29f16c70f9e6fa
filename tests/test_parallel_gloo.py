"""N > 1 host logic on CPU (gloo, world_size 2): slicing of the ensemble by the global trajectory index, the
histogram all-reduce and the rank-ordered image gather.  The per-rank compute is injected by the test as the oracle
(tests may call oracle/; the product itself has no CPU path), so what is checked is the plumbing: the sharded job
reproduces the single-process result EXACTLY — image bit for bit, histogram count for count — for the grid with
seeded angles, for a cloud (every rank draws its own slice of the random stream, not the same cloud twice) and for
both scaling modes.  The same bit-identity of the CUDA kernels on a slice is tests/test_gpu_parity_r2.py
(test_slices_are_bit_identical_to_the_whole)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

CASES = {
    # name: (gx, gy, shape, angle_mode, cx, cy, r, E, eps)
    "grid_angles0": (16, 10, 0, 0, 0.0, 0.0, 0.0, 1.0, 3e-2),
    "grid_seeded": (16, 11, 0, 1, 0.0, 0.0, 0.0, 1.0, 3e-2),
    "disk_cloud": (16, 9, 1, 1, 0.0, 0.0, 0.3, 1.0, 1e-3),
    "sphere": (8, 13, 3, 1, 0.0, 0.0, 0.0, 15.0, 1.0),
}


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _run(orc, gx, gy_total, k0, n, shape, angle_mode, cx, cy, r, E, eps, steps):
    st = orc.State(n, tangent=True, wind=True)
    g = orc.make_grid(gx, gy_total, -1.0, 1.0, angle_mode, shape, cx, cy, r, k0=k0)
    orc.init_shell(st, g, E, eps, 3)
    orc.integrate(st, steps, 0.005, 100)
    hist = np.zeros((64, 64), dtype=np.uint32)
    lim = 1.1 * (2 * E) ** 0.5
    orc.density(st, hist, -lim, lim)
    return orc.indicator(st, 0), hist


def _worker(rank, world, port, case, scaling, steps, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_1107_4107_b200 import parallel
    gx, gy, shape, angle_mode, cx, cy, r, E, eps = CASES[case]
    gxt, gyt, k0, n = parallel.slice_of(gx, gy, world, rank, scaling)
    fli, hist = _run(oracle, gxt, gyt, k0, n, shape, angle_mode, cx, cy, r, E, eps, steps)
    hist_t = torch.from_numpy(hist.view(np.int32).copy())
    parallel.allreduce_hist(hist_t)
    counts = [parallel.slice_of(gx, gy, world, rr, scaling)[3] for rr in range(world)]
    img = parallel.gather_image(torch.from_numpy(fli), counts)
    assert (img is None) == (rank != 0)
    if rank == 0:
        np.save(os.path.join(out_dir, "img.npy"), img.numpy())
    np.save(os.path.join(out_dir, "hist%d.npy" % rank), hist_t.numpy().view(np.uint32))
    dist.destroy_process_group()


@pytest.mark.parametrize("case,scaling", [("grid_angles0", "strong"), ("grid_seeded", "strong"), ("grid_seeded", "weak"),
                                          ("disk_cloud", "weak"), ("sphere", "strong")])
def test_sharded_job_equals_single_process_exactly(tmp_path, orc, case, scaling):
    world, steps = 2, 200
    mp.spawn(_worker, args=(world, _free_port(), case, scaling, steps, str(tmp_path)), nprocs=world, join=True)
    gx, gy, shape, angle_mode, cx, cy, r, E, eps = CASES[case]
    gy_total = gy * world if scaling == "weak" else gy
    ref_img, ref_hist = _run(orc, gx, gy_total, 0, gx * gy_total, shape, angle_mode, cx, cy, r, E, eps, steps)
    img = np.load(tmp_path / "img.npy")
    assert img.shape == ref_img.shape
    assert np.array_equal(img, ref_img, equal_nan=True)            # bit for bit, NaN pixels in the same places
    h0, h1 = np.load(tmp_path / "hist0.npy"), np.load(tmp_path / "hist1.npy")
    assert np.array_equal(h0, h1) and np.array_equal(h0, ref_hist)
    assert h0.sum() > 0


def test_ranks_of_a_cloud_draw_different_slices(orc):
    """The defect this replaces: every rank seeding the same cloud.  Two ranks' slices of a seeded ensemble differ."""
    from paper_1107_4107_b200 import parallel
    a = parallel.slice_of(16, 9, 2, 0, "weak")
    b = parallel.slice_of(16, 9, 2, 1, "weak")
    assert a == (16, 18, 0, 144) and b == (16, 18, 144, 144)
    sa = orc.init_shell(orc.State(144), orc.make_grid(16, 18, angle_mode=1, shape=1, r=0.3, k0=a[2]), 1.0, 1e-3, 3)
    sb = orc.init_shell(orc.State(144), orc.make_grid(16, 18, angle_mode=1, shape=1, r=0.3, k0=b[2]), 1.0, 1e-3, 3)
    assert not np.array_equal(sa.q[:, :144], sb.q[:, :144])


def test_shard_rows_and_slices():
    from paper_1107_4107_b200 import parallel
    for gy in (1, 7, 2048, 2049):
        for world in (1, 2, 3, 8):
            edges = [parallel.shard_rows(gy, world, r) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == gy
            assert all(a[1] == b[0] for a, b in zip(edges[:-1], edges[1:]))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1
            sl = [parallel.slice_of(5, gy, world, r, "strong") for r in range(world)]
            assert sum(s[3] for s in sl) == 5 * gy and sl[0][2] == 0
            assert all(a[2] + a[3] == b[2] for a, b in zip(sl[:-1], sl[1:]))
            assert all(s[:2] == (5, gy) for s in sl)
            wk = [parallel.slice_of(5, gy, world, r, "weak") for r in range(world)]
            assert all(s == (5, gy * world, r * 5 * gy, 5 * gy) for r, s in enumerate(wk))
    with pytest.raises(ValueError):
        parallel.shard_rows(8, 2, 2)
    with pytest.raises(ValueError):
        parallel.slice_of(8, 8, 2, 0, "diagonal")


def test_allreduce_hist_uint32_wraparound_semantics():
    """int32 two's-complement addition carries the uint32 bits exactly (counts above 2^31)."""
    a = np.array([0x7fffffff, 0xfffffff0, 5], dtype=np.uint32)
    b = np.array([1, 0x0f, 7], dtype=np.uint32)
    s = (torch.from_numpy(a.view(np.int32).copy()) + torch.from_numpy(b.view(np.int32).copy())).numpy().view(np.uint32)
    assert np.array_equal(s, (a.astype(np.uint64) + b).astype(np.uint32))

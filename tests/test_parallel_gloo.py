"""N > 1 host logic on CPU (gloo, world_size 2): row sharding, strip bounds, the histogram all-reduce
and the rank-ordered image gather.  The per-rank compute is injected by the test as the oracle (tests may
call oracle/; the product itself has no CPU path), so what is checked is the plumbing: the sharded job
reproduces the single-process result exactly."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, gx, gy, steps, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_1107_4107_b200 import parallel
    j0, j1 = parallel.shard_rows(gy, world, rank)
    rows = j1 - j0
    # rank-local strip of the image: same cell centres as the corresponding rows of the whole grid
    h = 2.0 / gy
    st = oracle.State(gx * rows, tangent=True, wind=True)
    g = oracle.make_grid(gx, rows, -1.0, 1.0, angle_mode=0, lo_y=-1.0 + j0 * h, hi_y=-1.0 + j1 * h)
    oracle.init_shell(st, g, 1.0, 3e-2, 0)
    oracle.integrate(st, steps, 0.005, 100)
    fli = torch.from_numpy(oracle.indicator(st, 0).reshape(rows, gx))
    hist = np.zeros((64, 64), dtype=np.uint32)
    oracle.density(st, hist, -1.0, 1.0)
    hist_t = torch.from_numpy(hist.view(np.int32).copy())
    parallel.allreduce_hist(hist_t)
    img = parallel.gather_image(fli, world, rank)
    if rank == 0:
        np.save(os.path.join(out_dir, "img.npy"), img.numpy())
    np.save(os.path.join(out_dir, "hist%d.npy" % rank), hist_t.numpy().view(np.uint32))
    dist.destroy_process_group()


def test_sharded_job_equals_single_process(tmp_path, orc):
    gx, gy, steps, world = 16, 10, 300, 2
    mp.spawn(_worker, args=(world, _free_port(), gx, gy, steps, str(tmp_path)), nprocs=world, join=True)
    st = orc.State(gx * gy, tangent=True, wind=True)
    orc.init_shell(st, orc.make_grid(gx, gy, -1.0, 1.0), 1.0, 3e-2, 0)
    orc.integrate(st, steps, 0.005, 100)
    ref_img = orc.indicator(st, 0).reshape(gy, gx)
    ref_hist = np.zeros((64, 64), dtype=np.uint32)
    orc.density(st, ref_hist, -1.0, 1.0)
    img = np.load(tmp_path / "img.npy")
    # strips use lo_y + (j + 1/2) h with their own lo_y: cell centres agree with the whole grid to rounding
    assert img.shape == ref_img.shape
    assert np.allclose(img, ref_img, rtol=0, atol=1e-9, equal_nan=True)
    h0, h1 = np.load(tmp_path / "hist0.npy"), np.load(tmp_path / "hist1.npy")
    assert np.array_equal(h0, h1)
    assert h0.sum() == ref_hist.sum() == (st.status == 1).sum()
    assert np.abs(h0.astype(np.int64) - ref_hist.astype(np.int64)).sum() <= 4   # cell-centre rounding only


def test_shard_rows_and_strip_bounds():
    from paper_1107_4107_b200 import parallel
    for gy in (1, 7, 2048, 2049):
        for world in (1, 2, 3, 8):
            edges = [parallel.shard_rows(gy, world, r) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == gy
            assert all(a[1] == b[0] for a, b in zip(edges[:-1], edges[1:]))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1
    for world in (1, 2, 4, 8):
        b = [parallel.strip_bounds(-1.0, 1.0, world, r) for r in range(world)]
        assert b[0][0] == -1.0 and b[-1][1] == 1.0
        assert all(x[1] == y[0] for x, y in zip(b[:-1], b[1:]))
    with pytest.raises(ValueError):
        parallel.strip_bounds(-1.0, 1.0, 2, 2)


def test_allreduce_hist_uint32_wraparound_semantics():
    """int32 two's-complement addition carries the uint32 bits exactly (counts above 2^31)."""
    a = np.array([0x7fffffff, 0xfffffff0, 5], dtype=np.uint32)
    b = np.array([1, 0x0f, 7], dtype=np.uint32)
    s = (torch.from_numpy(a.view(np.int32).copy()) + torch.from_numpy(b.view(np.int32).copy())).numpy().view(np.uint32)
    assert np.array_equal(s, (a.astype(np.uint64) + b).astype(np.uint32))

"""Multi-GPU host logic on CPU: batch sharding and the max-over-ranks reduction, world_size 2 over gloo."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1503_05768_b200.shard import max_over_ranks, shard_range, sum_over_ranks


def test_shard_range_partitions_exactly():
    for n in (0, 1, 2, 7, 128, 129):
        for world in (1, 2, 3, 4, 8):
            spans = [shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            for (a0, a1), (b0, b1) in zip(spans, spans[1:]):
                assert a1 == b0 and a1 >= a0
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = shard_range(128, rank, world)
    dist.barrier()
    t = max_over_ranks(1.0 + rank)            # slowest rank decides
    n = sum_over_ranks(hi - lo)               # units all ranks processed
    q.put((rank, lo, hi, t, n))
    dist.destroy_process_group()


def test_world_size_2_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [(r[1], r[2]) for r in res] == [(0, 64), (64, 128)]
    assert all(r[3] == 2.0 and r[4] == 128.0 for r in res)


def test_single_process_is_identity():
    assert max_over_ranks(3.5) == 3.5 and sum_over_ranks(7) == 7.0
    assert isinstance(torch.tensor([1.0]).item(), float)


# ---- one large image split into row slabs with a 2 r T overlap (no exchange): host logic with the oracle as the compute ----
def _slab_worker(rank, world, port, q):
    import numpy as np
    import oracle
    import tnrd_gen
    from paper_1503_05768_b200.shard import slab_bounds
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    c = tnrd_gen.make_small(81, 1, 90, 40, 2, 3, 5)
    H = c["H"]
    lo, hi, s0, s1 = slab_bounds(H, rank, world, c["T"], c["ksize"])
    part = oracle.diffuse(c["f"][:, s0:s1], c["u0"][:, s0:s1], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"],
                          c["lambda"])[:, lo - s0:hi - s0]
    rows = torch.zeros((H, c["W"]), dtype=torch.float64)
    rows[lo:hi] = torch.from_numpy(part[0])
    dist.all_reduce(rows)                      # test-side stitching only; the product path has no collective
    if rank == 0:
        full = oracle.diffuse(c["f"], c["u0"], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], c["lambda"])[0]
        q.put(float(np.max(np.abs(rows.numpy() - full))))
    dist.destroy_process_group()


def test_row_slabs_with_overlap_reproduce_the_full_image_world_size_2_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_slab_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    err = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert err == 0.0                          # the slab's interior is bit-identical to the full image (locality)


def test_slab_bounds():
    from paper_1503_05768_b200.shard import slab_bounds
    assert slab_bounds(4096, 0, 8, 5, 7) == (0, 512, 0, 542)
    assert slab_bounds(4096, 3, 8, 5, 7) == (1536, 2048, 1506, 2078)
    assert slab_bounds(4096, 7, 8, 5, 7) == (3584, 4096, 3554, 4096)
    assert slab_bounds(10, 1, 2, 8, 9) == (5, 10, 0, 10)

"""Host logic of the sharded operator (paper_2503_06721_b200/slab.py) on CPU: partition arithmetic and, with two gloo
processes, the face exchange pattern (who receives which slice).  No GPU, no kernels."""
import os
import socket

import numpy as np
import pytest

from paper_2503_06721_b200 import slab


def test_partition_is_even_contiguous_and_complete():
    for T, w in [(8, 1), (8, 2), (8, 4), (12, 2), (20, 3), (96, 8), (32, 5)]:
        parts = slab.partition(T, w)
        assert len(parts) == w and parts[0][0] == 0 and sum(n for _, n in parts) == T
        for (t0, n0), (t1, _) in zip(parts, parts[1:]):
            assert t0 + n0 == t1
        assert all(t % 2 == 0 and n % 2 == 0 and n >= 2 for t, n in parts)
        assert max(n for _, n in parts) - min(n for _, n in parts) <= 2
    for bad in [(7, 2), (4, 3), (8, 0)]:
        with pytest.raises(ValueError):
            slab.partition(*bad)
    assert slab.neighbours(0, 4) == (3, 1) and slab.neighbours(3, 4) == (2, 0) and slab.neighbours(0, 1) == (0, 0)


def _worker(rank, world, port, T, S, q):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        field = torch.arange(T * S, dtype=torch.float64).reshape(T, S)      # "global" field: value identifies (slice, site)
        t0, n = slab.partition(T, world)[rank]
        first, last = field[t0].clone(), field[t0 + n - 1].clone()
        from_next, from_prev = torch.empty(S, dtype=torch.float64), torch.empty(S, dtype=torch.float64)
        slab.exchange_faces(dist, rank, world, first, last, from_next, from_prev)
        ok = bool(torch.equal(from_next, field[(t0 + n) % T]) and torch.equal(from_prev, field[(t0 - 1) % T]))
        q.put((rank, ok))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,T", [(2, 8), (2, 4)])
def test_face_exchange_gloo(world, T):
    """Each rank must end up with the slice after its last owned one (from the next rank) and the slice before its first (from the
    previous rank), periodically -- the ghost slices of hirep_geom_create_slab."""
    import torch.multiprocessing as mp
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, T, 24, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
    assert sorted(res) == [(r, True) for r in range(world)]


def test_exchange_single_rank_wraps():
    import torch
    a, b = torch.arange(4.0), torch.arange(4.0) + 10
    rn, rp = torch.empty(4), torch.empty(4)
    slab.exchange_faces(None, 0, 1, a, b, rn, rp)
    assert torch.equal(rn, a) and torch.equal(rp, b)

"""N > 1 host logic on CPU: two gloo processes shard a batch of specimens, time reduction is the max over ranks
(no data-path collective; replicas or specimen shards)."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2201_04565_b200.multi import reduce_over_ranks, shard_units
from lsm_inputs import config4


def test_shard_units_partitions_exactly():
    for n in (0, 1, 5, 7, 1024, 1025):
        for world in (1, 2, 3, 8):
            parts = [shard_units(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[r][1] == parts[r + 1][0] for r in range(world - 1))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_units(4, 2, 2)


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        B, n = 5, 12
        lo, hi = shard_units(B, rank, world)
        p = config4(B=hi - lo, n=n, first=lo)            # this rank's specimens, as bench.py builds them
        # per-rank "device time" and work done; value = all units / max time
        t_ms, units = 10.0 * (rank + 1), float(p.M)
        tmax, = reduce_over_ranks([t_ms], "max", dist)
        usum, = reduce_over_ranks([units], "sum", dist)
        dist.barrier()
        q.put((rank, lo, hi, p.N, p.M, float(p.x.sum()), float(p.k.sum()), tmax, usum))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_shard_config4_and_reduce():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for pr in procs:
        pr.start()
    out = sorted(q.get(timeout=120) for _ in range(2))
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    full = config4(B=5, n=12)
    (r0, lo0, hi0, N0, M0, sx0, sk0, tmax0, usum0), (r1, lo1, hi1, N1, M1, sx1, sk1, tmax1, usum1) = out
    assert (lo0, hi0, lo1, hi1) == (0, 3, 3, 5)
    assert N0 + N1 == full.N and M0 + M1 == full.M                 # shards cover the batch exactly once
    assert np.isclose(sk0 + sk1, full.k.sum(), rtol=1e-13) and np.isclose(sx0 + sx1, full.x.sum(), rtol=1e-12)
    assert tmax0 == tmax1 == 20.0 and usum0 == usum1 == float(full.M)   # max over ranks, whole-job units

"""N > 1 host logic on CPU: world_size-2 gloo run of id sharding + tally reduction.  Each rank tracks its id
range with the ORACLE (tests may call it); the reduced tally must equal a single-process run bit-for-bit in the
counts and to rounding in the sums."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out_path):
    sys.path.insert(0, ROOT); sys.path.insert(0, os.path.join(ROOT, "tests"))
    from oracle_binding import Oracle
    from paper_2602_13198_b200 import workloads as wl
    from paper_2602_13198_b200.shard import id_range, reduce_tally
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    p, prim = wl.config1(Ns=4e3)
    o = Oracle(p, prim)
    n = o.prepare()
    first, cnt = id_range(n, rank, world)
    o.run(first, cnt, 1)
    ts = [torch.from_numpy(np.ascontiguousarray(a)) for a in o.tally()]
    reduce_tally(ts, dist)
    if rank == 0:
        np.savez(out_path, A=ts[0].numpy(), Q=ts[1].numpy(), W=ts[2].numpy(), n=ts[3].numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_id_ranges_tile_exactly():
    from paper_2602_13198_b200.shard import id_range, rank_seed
    for n in (0, 1, 7, 1000, 12345):
        for world in (1, 2, 3, 8):
            r = [id_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and sum(c for _, c in r) == n
            for (f0, c0), (f1, _) in zip(r, r[1:]):
                assert f0 + c0 == f1
    assert rank_seed(1, 0) == 1 and len({rank_seed(1, k) for k in range(64)}) == 64


def test_two_rank_sharded_run_equals_single_run(tmp_path):
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from oracle_binding import Oracle
    from paper_2602_13198_b200 import workloads as wl
    out = str(tmp_path / "t.npz")
    mp.spawn(_worker, args=(2, 29500 + os.getpid() % 2000, out), nprocs=2, join=True)
    got = np.load(out)
    p, prim = wl.config1(Ns=4e3)
    o = Oracle(p, prim); o.prepare(); o.run(nthreads=1)
    A, Q, W, n = o.tally()
    assert np.array_equal(got["n"], n)
    assert np.allclose(got["A"], A, rtol=1e-12, atol=0) and np.allclose(got["W"], W, rtol=1e-12, atol=0)

"""The N > 1 path on CPU: two `gloo` ranks (task statement (5)).

The path shards by contiguous particle ranges with no data-path collective; the one exchange a
distributed bunch needs is the monitor record, merged from the per-rank records by `hb_moments_merge`
(host arithmetic inside libhb.so) after an all-gather of 27 doubles + a count per monitor.  No GPU is needed for
any of that, so here each rank produces its shard's record with the fp64 oracle (which tests may call), the product's
`allgather_merge_records` merges them over gloo, and the result is compared with the oracle's record of the whole
bunch.  Also covered: the shard ranges two ranks derive are disjoint and cover the bunch; the max-over-ranks
reduction bench.py uses for its time.
"""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n, q):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch
    import torch.distributed as dist
    import oracle
    import workloads as wl
    import paper_2402_17248_b200 as hb
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # every rank draws the same seeded bunch and a two-monitor lattice, then keeps only its own range
        desc = wl.lattice([wl.drift(0.7), wl.quad(0.3, 4.0), wl.monitor(), wl.drift(1.1), wl.quad(0.3, -4.0),
                           wl.monitor()])
        x = wl.gaussian_bunch(n, seed=31)
        lo, hi = wl.shard_range(n, rank, world)
        _, rec_local = oracle.push(desc, np.ascontiguousarray(x[:, lo:hi].astype(np.float64)))
        merged = hb.allgather_merge_records(rec_local, hi - lo)
        _, rec_global = oracle.push(desc, np.ascontiguousarray(x.astype(np.float64)))
        # all ranks hold identical bytes (merge order is rank order everywhere)
        mine = torch.from_numpy(merged.copy())
        parts = [torch.empty_like(mine) for _ in range(world)]
        dist.all_gather(parts, mine)
        same = all(torch.equal(parts[0], p) for p in parts)
        # bench.py's timing reduction: max over ranks
        t = torch.tensor([float(rank + 1)], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        q.put((rank, lo, hi, merged, np.asarray(rec_global), same, float(t[0])))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n", [10_001, 3])
def test_two_gloo_ranks_reproduce_the_global_monitor_records(n):
    import torch.multiprocessing as mp
    from paper_2402_17248_b200.build import build_lib
    build_lib()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=240) for _ in procs], key=lambda r: r[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, lo0, hi0, m0, g0, same0, t0), (_, lo1, hi1, m1, g1, same1, t1) = res
    assert lo0 == 0 and hi0 == lo1 and hi1 == n
    assert same0 and same1 and np.array_equal(m0, m1)
    assert t0 == 2.0 and t1 == 2.0
    assert m0.shape == g0.shape == (2, 27)
    diag = [6, 12, 17, 21, 24, 26]
    for k in range(2):
        assert np.allclose(m0[k][:6], g0[k][:6], rtol=1e-12, atol=1e-18)
        scale = np.sqrt(np.outer(g0[k][diag], g0[k][diag]))[np.triu_indices(6)]
        assert np.all(np.abs(m0[k][6:] - g0[k][6:]) <= 1e-12 * scale)

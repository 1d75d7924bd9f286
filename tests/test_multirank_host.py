"""N > 1 path of bench.py on CPU: world_size-2 gloo processes exercise the rank bookkeeping
(per-rank right-hand sides, MAX-over-ranks time, SUM of iterations).  The data path itself has
no collective (replicas only)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    w, dtype, fmt = bench.make_workload("config4_small_c128_bsr3", rank, want_csr=False)
    # each rank "measures" a different time and iteration count
    (t_max, t2), (iters, launches) = bench.aggregate_over_ranks([10.0 + 5.0 * rank, 1.0], [24 + rank, 100], "cpu", world)
    out[rank] = (t_max, iters, launches, complex(w.b[0]), bench.throughput(iters, t_max))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_aggregation_gloo():
    world = 2
    port = _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    r0, r1 = out[0], out[1]
    assert r0[0] == r1[0] == 15.0                 # MAX over ranks
    assert r0[1] == r1[1] == 49.0                 # SUM of iterations
    assert r0[2] == 200.0
    assert r0[3] != r1[3]                         # replicas solve different right-hand sides
    assert np.isclose(r0[4], 49.0 / 15e-3)


def test_single_rank_passthrough():
    import bench
    (t,), (c,) = bench.aggregate_over_ranks([3.0], [7], "cpu", 1)
    assert t == 3.0 and c == 7.0


def _shard_worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import oracle
    from paper_1102_2143_b200 import workloads as W
    w = W.config2(extents=(4, 4, 4, 4))
    mine = bench.shard_shifts(w.shifts, rank, world)
    res = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, mine, w.tol, w.max_iter)
    # the job's iteration count under --shard shifts: MAX over ranks of the per-rank counts
    (it_max,), _ = bench.aggregate_over_ranks([float(res.iterations)], [0], "cpu", world)
    out[rank] = (mine.copy(), res.x.copy(), res.conv_iter.copy(), res.iterations, it_max)
    dist.barrier()
    dist.destroy_process_group()


def test_shift_sharding_two_ranks_gloo():
    """bench.py --shard shifts: the ranks split the shifts of ONE system with no collective on the data
    path.  The oracle shows why that is exact: every x_k depends on the base Krylov sequence only
    (PAPER.md:47-57), so each rank's solutions are bit-identical to the full solve's."""
    import oracle
    from paper_1102_2143_b200 import workloads as W
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_shard_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    w = W.config2(extents=(4, 4, 4, 4))
    full = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, w.shifts, w.tol, w.max_iter)
    seen = []
    for r in range(world):
        mine, x, conv, its, it_max = out[r]
        assert it_max == full.iterations == max(out[q][3] for q in range(world))
        for j, s in enumerate(mine):
            k = int(np.where(w.shifts == s)[0][0])
            seen.append(k)
            assert np.array_equal(x[j], full.x[k])            # bitwise: shifts do not interact
            assert conv[j] == full.conv_iter[k]
    assert sorted(seen) == list(range(w.shifts.size))          # disjoint cover of the family

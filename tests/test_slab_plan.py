"""Row partition, host side: the halo plan of msolve_slab_plan_* (no GPU).

Single process: the plans of all slabs of a matrix against what the matrix itself says (every off-slab column of
every slab row is covered exactly once, the renumbered columns reproduce the global ones, a slab SpMV in numpy
on [own | halo] vectors reproduces the rows of the global product).
Two gloo ranks: each rank builds the plan of ITS slab only, the ranks exchange their receive lists (what a
multi-process run does once at set-up) and check the send side against them."""
import os
import socket

import numpy as np
import pytest
import scipy.sparse as sp
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1102_2143_b200 import workloads as W


def _plan(n, splits, rank, rowptr, colidx):
    from paper_1102_2143_b200 import binding, build
    build.build()
    rb, re = splits[rank], splits[rank + 1]
    rp = (rowptr[rb:re + 1] - rowptr[rb]).astype(np.int32)
    return binding.SlabPlan(n, splits, rank, rp, colidx[rowptr[rb]:rowptr[re]])


def _check_slab(w_rowptr, w_colidx, n, splits, rank, plan):
    rb, re = splits[rank], splits[rank + 1]
    cols = w_colidx[w_rowptr[rb]:w_rowptr[re]]
    off = np.unique(cols[(cols < rb) | (cols >= re)])
    # every off-slab column exactly once, grouped by owner ascending, ascending within an owner
    ids = np.concatenate([p[2] for p in plan.peers]) if plan.peers else np.zeros(0, np.int32)
    assert plan.nlocal == re - rb and plan.nhalo == off.size == ids.size
    assert np.array_equal(ids, off)
    pos = 0
    for peer, offset, gid in plan.peers:
        assert peer != rank and offset == pos and gid.size > 0
        assert np.all((gid >= splits[peer]) & (gid < splits[peer + 1]))
        pos += gid.size
    assert [p[0] for p in plan.peers] == sorted(set(p[0] for p in plan.peers))
    # renumbered columns give back the global ones
    back = np.where(plan.colidx < plan.nlocal, plan.colidx + rb, ids[np.maximum(plan.colidx - plan.nlocal, 0)] if ids.size else 0)
    assert np.array_equal(back, cols)


@pytest.mark.parametrize("which", ["lattice", "powerlaw", "poisson"])
@pytest.mark.parametrize("nslabs", [1, 2, 3, 8])
def test_plans_cover_every_off_slab_column_once(which, nslabs):
    w = {"lattice": lambda: W.config2(extents=(4, 4, 4, 8)), "powerlaw": lambda: W.config5(n=3001),
         "poisson": lambda: W.poisson_workload(23, 17, real=True)}[which]()
    n = w.n
    splits = np.array([n * p // nslabs for p in range(nslabs + 1)], dtype=np.int64)
    A = sp.csr_matrix((w.val, w.colidx, w.rowptr), shape=(n, n))
    rng = np.random.default_rng(2)
    x = rng.standard_normal(n) + (0 if np.isrealobj(w.val) else 1j * rng.standard_normal(n))
    y = A @ x
    for rank in range(nslabs):
        plan = _plan(n, splits, rank, w.rowptr, w.colidx)
        _check_slab(w.rowptr, w.colidx, n, splits, rank, plan)
        # the slab's product from its own rows and an [own | halo] vector
        rb, re = splits[rank], splits[rank + 1]
        ids = np.concatenate([p[2] for p in plan.peers]) if plan.peers else np.zeros(0, np.int64)
        xext = np.concatenate([x[rb:re], x[ids]])
        rp = w.rowptr[rb:re + 1] - w.rowptr[rb]
        Aloc = sp.csr_matrix((w.val[w.rowptr[rb]:w.rowptr[re]], plan.colidx, rp), shape=(re - rb, xext.size))
        assert np.allclose(Aloc @ xext, y[rb:re], rtol=0, atol=1e-12 * np.abs(y).max())


def test_plan_validation():
    from paper_1102_2143_b200 import binding, build
    build.build()
    rp = np.array([0, 1, 2], dtype=np.int32)
    with pytest.raises(binding.MsolveError):                       # splits do not end at n
        binding.SlabPlan(4, [0, 2, 3], 0, rp, np.array([0, 1], dtype=np.int32))
    with pytest.raises(binding.MsolveError):                       # column out of range
        binding.SlabPlan(4, [0, 2, 4], 0, rp, np.array([0, 4], dtype=np.int32))
    with pytest.raises(binding.MsolveError):                       # rank out of range
        binding.SlabPlan(4, [0, 2, 4], 2, rp, np.array([0, 1], dtype=np.int32))
    p = binding.SlabPlan(4, [0, 2, 4], 1, rp, np.array([0, 3], dtype=np.int32))     # slab 1 = rows 2, 3
    assert p.nlocal == 2 and p.nhalo == 1 and p.peers[0][0] == 0 and p.peers[0][2].tolist() == [0]
    assert p.colidx.tolist() == [2, 1]
    e = binding.SlabPlan(4, [0, 4, 4], 1, np.array([0], dtype=np.int32), np.zeros(0, dtype=np.int32))   # empty slab
    assert e.nlocal == 0 and e.nhalo == 0 and not e.peers


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.config4(extents=(4, 4, 4, 8), want_csr=True)                 # split along t, as config 4 would be
    n = w.n
    splits = np.array([n * p // world for p in range(world + 1)], dtype=np.int64)
    plan = _plan(n, splits, rank, w.rowptr, w.colidx)                   # this rank's slab only
    mine = {peer: gid.tolist() for peer, _, gid in plan.peers}          # what I receive, from whom
    everyone = [None] * world
    dist.all_gather_object(everyone, mine)                              # set-up exchange of the receive lists
    # my send lists = the others' receive lists that name me; every id must be one of MY rows
    send = {q: everyone[q].get(rank, []) for q in range(world) if q != rank}
    ok = all(splits[rank] <= g < splits[rank + 1] for ids in send.values() for g in ids)
    out[rank] = (plan.nlocal, plan.nhalo, mine, send, ok)
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_halo_lists_gloo():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    w = W.config4(extents=(4, 4, 4, 8), want_csr=True)
    n = w.n
    assert out[0][0] + out[1][0] == n and out[0][4] and out[1][4]
    for r in range(world):
        q = 1 - r
        # what r sends to q is exactly what q receives from r, in the same order
        assert out[r][3][q] == out[q][2].get(r, [])
        # periodic lattice split along t: each slab needs the two boundary time slices of the other
        # (4^3 sites x 3 colours each), i.e. 2 x 192 halo elements
        assert out[r][1] == 2 * 4 * 4 * 4 * 3

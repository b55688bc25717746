"""NEXT-4, multi-rank host logic on CPU (world size 2 and 3, gloo): the interface plan and the pairwise exchange of
paper_2110_01716_b200/sharded.py, driven with HOST buffers.  Each rank computes its rank-local w with the oracle (the
CUDA kernels cannot run here), packs / exchanges / adds exactly as ShardedSem does on the GPU, and the result is compared
with the oracle's single-rank M QQ^T A_L u: bit-identical on nodes that live on one rank only, 1e-12 on interface nodes."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    sys.path.insert(0, ROOT)
    import oracle
    from paper_2110_01716_b200 import inputs, sharded
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        m = inputs.box_mesh(4, 3, 3, 4, "random", seed=8, permute_seed=2)      # scrambled element order: ragged interfaces
        b = sharded.partition_bounds(m.E, world)
        sl = slice(b[rank], b[rank + 1])
        gid, vert, dirf = m.gid[sl], m.vert[sl], m.dirichlet[sl]
        comm = sharded.DistComm()
        cand = comm.all_gather_arrays(sharded.surface_gids(gid, m.N))
        plan = sharded.interface_plan(rank, cand)
        # rank-local operator + rank-local gather-scatter + mask (the oracle stands in for sem_ax_gs here)
        om = oracle.Maps(gid)
        G, _, rc = oracle.geom_trilinear(vert, m.N)
        assert rc == 0
        u = inputs.field_uniform(gid, 12)
        mask_l = oracle.mask_unique(dirf, om)[om.l2u] != 0
        w = np.where(mask_l, 0.0, oracle.gs(oracle.ax(G, u, m.N).ravel(), om))
        # pack (first copy), exchange, add to every copy in ascending rank order: what sem_iface_pack / _add do
        uniq = {r: np.searchsorted(om.uniq_gid, g) for r, g in plan.items()}
        send = {r: torch.from_numpy(w[om.seg_idx[om.seg_off[q]]].copy()) for r, q in uniq.items()}
        recv = {r: torch.empty_like(t) for r, t in send.items()}
        comm.exchange(send, recv)
        mask_u = oracle.mask_unique(dirf, om)
        for r in sorted(uniq):
            for q, v in zip(uniq[r], recv[r].numpy()):
                if not mask_u[q]:
                    w[om.seg_idx[om.seg_off[q]:om.seg_off[q + 1]]] += v
        shared_local = np.zeros(om.U, bool)
        for q in uniq.values():
            shared_local[q] = True
        out[rank] = (b[rank], b[rank + 1], w, shared_local[om.l2u], {r: len(g) for r, g in plan.items()})
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_apply_matches_single_rank(world):
    sys.path.insert(0, ROOT)
    import oracle
    from paper_2110_01716_b200 import inputs
    oracle.build()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    m = inputs.box_mesh(4, 3, 3, 4, "random", seed=8, permute_seed=2)
    om = oracle.Maps(m.gid)
    G, _, _ = oracle.geom_trilinear(m.vert, m.N)
    u = inputs.field_uniform(m.gid, 12)
    mask_l = oracle.mask_unique(m.dirichlet, om)[om.l2u] != 0
    ref = np.where(mask_l, 0.0, oracle.gs(oracle.ax(G, u, m.N).ravel(), om)).reshape(m.E, -1)
    scale = np.max(np.abs(ref))
    n_iface = 0
    for rank in range(world):
        lo, hi, w, shared, sizes = res[rank]
        w = w.reshape(hi - lo, -1)
        shared = shared.reshape(hi - lo, -1)
        assert np.array_equal(w[~shared], ref[lo:hi][~shared])                  # one rank only: bit-identical
        assert np.max(np.abs(w - ref[lo:hi])) <= 1e-12 * scale                  # interface: round-off
        n_iface += int(shared.sum())
        for r, n in sizes.items():                                              # symmetric plan
            assert res[r][4][rank] == n
    assert n_iface > 0


def _pcg_worker(rank: int, world: int, port: int, out):
    """The recurrence of sem_pcg_sharded (include/sem.h) on host arrays, the oracle standing in for the rank-local
    kernels: interface-first element order, exchange started and finished separately, global dot weights and Jacobi
    diagonal through the exchange, two all-reduces per iteration."""
    sys.path.insert(0, ROOT)
    import oracle
    from paper_2110_01716_b200 import inputs, sharded
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        m = inputs.box_mesh(4, 3, 3, 3, "random", seed=8, permute_seed=2)
        b = sharded.partition_bounds(m.E, world)
        sl = slice(b[rank], b[rank + 1])
        comm = sharded.DistComm()
        plan = sharded.interface_plan(rank, comm.all_gather_arrays(sharded.surface_gids(m.gid[sl], m.N)))
        flagged = comm.all_gather_arrays(np.unique(m.gid[sl][m.dirichlet[sl] != 0]))
        sharded.check_mask_agreement(rank, plan, flagged)
        perm, n_iface = sharded.interface_first(m.gid[sl], plan)
        gid, vert, dirf = m.gid[sl][perm], m.vert[sl][perm], m.dirichlet[sl][perm]
        shared_all = np.unique(np.concatenate(list(plan.values())))
        touches = np.isin(gid.reshape(len(gid), -1), shared_all).any(axis=1)
        assert touches[:n_iface].all() and not touches[n_iface:].any()
        om = oracle.Maps(gid)
        G, _, _ = oracle.geom_trilinear(vert, m.N)
        mask_u = oracle.mask_unique(dirf, om)
        live = (mask_u == 0)[om.l2u]
        uniq = {r: np.searchsorted(om.uniq_gid, g) for r, g in plan.items()}
        first = om.seg_idx[om.seg_off[:-1]]

        def gs_across(w):
            send = {r: torch.from_numpy(w[first[q]].copy()) for r, q in uniq.items()}
            recv = {r: torch.empty_like(t) for r, t in send.items()}
            handle = comm.start_exchange(send, recv)
            comm.finish_exchange(handle)
            add_u = np.zeros(om.U)
            for r in sorted(uniq):
                add_u[uniq[r]] += np.where(mask_u[uniq[r]] != 0, 0.0, recv[r].numpy())
            return w + add_u[om.l2u]

        def A(p):
            return gs_across(np.where(live, oracle.gs(oracle.ax(G, p.reshape(len(gid), -1), m.N).ravel(), om), 0.0))

        def allsum(*v):
            t = torch.tensor(v, dtype=torch.float64)
            comm.allreduce(t)
            return t.tolist()

        mult_g = gs_across(om.mult[om.l2u].astype(np.float64))
        diag_g = gs_across(oracle.gs(oracle.diag_local(G, m.N).ravel(), om))
        wt = np.where(live, 1.0 / mult_g, 0.0)
        Minv = np.where(live, 1.0 / diag_g, 0.0)
        # right-hand side: the whole-mesh b = A x*, restricted to this rank (computed by every rank from the seed)
        omw = oracle.Maps(m.gid)
        Gw, _, _ = oracle.geom_trilinear(m.vert, m.N)
        maskw = oracle.mask_unique(m.dirichlet, omw)
        xs = np.where(maskw != 0, 0.0, inputs.field_normal(omw.uniq_gid, 5))
        b_u = oracle.apply_Ag(Gw, m.N, omw, maskw, xs)
        bl = b_u[omw.l2u].reshape(m.E, -1)[sl][perm].ravel()
        x = np.zeros_like(bl)
        r_ = np.where(live, bl, 0.0)
        z = Minv * r_
        p = z.copy()
        rr0, rz = allsum(float(np.sum(wt * r_ * r_)), float(np.sum(wt * r_ * z)))
        hist, it = [1.0], 0
        for it in range(1, 301):
            q = A(p)
            (pq,) = allsum(float(np.sum(p * oracle.ax(G, p.reshape(len(gid), -1), m.N).ravel())))
            alpha = rz / pq
            x += alpha * p
            r_ -= alpha * q
            rr, rz_new = allsum(float(np.sum(wt * r_ * r_)), float(np.sum(wt * r_ * Minv * r_)))
            hist.append(np.sqrt(rr / rr0))
            if rr <= 1e-18 * rr0:
                break
            p = Minv * r_ + (rz_new / rz) * p
            rz = rz_new
        inv = np.empty_like(perm)
        inv[perm] = np.arange(len(perm))
        out[rank] = (b[rank], b[rank + 1], x.reshape(len(gid), -1)[inv], it, hist, n_iface)
    finally:
        dist.destroy_process_group()


def test_sharded_pcg_recurrence_gloo():
    sys.path.insert(0, ROOT)
    import oracle
    from paper_2110_01716_b200 import inputs
    oracle.build()
    world = 2
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_pcg_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    m = inputs.box_mesh(4, 3, 3, 3, "random", seed=8, permute_seed=2)
    om = oracle.Maps(m.gid)
    G, _, _ = oracle.geom_trilinear(m.vert, m.N)
    mask_u = oracle.mask_unique(m.dirichlet, om)
    xs = np.where(mask_u != 0, 0.0, inputs.field_normal(om.uniq_gid, 5))
    b_u = oracle.apply_Ag(G, m.N, om, mask_u, xs)
    ores = oracle.pcg(G, m.N, om, mask_u, b_u, tol=1e-9, maxit=300)
    xref = ores["x"][om.l2u].reshape(m.E, -1)
    for rank in range(world):
        lo, hi, x, it, hist, n_iface = res[rank]
        assert it == ores["iters"] and it == res[0][3] and hist == res[0][4]     # same decisions on every rank
        assert np.max(np.abs(x - xref[lo:hi])) <= 1e-8 * np.max(np.abs(xref))
        h = np.asarray(hist)
        big = ores["hist"] >= 1e-5
        assert np.max(np.abs(h[big] - ores["hist"][big]) / ores["hist"][big]) <= 1e-6
        assert 0 < n_iface <= hi - lo


def test_interface_first_and_mask_agreement():
    sys.path.insert(0, ROOT)
    from paper_2110_01716_b200 import inputs, sharded
    m = inputs.box_mesh(3, 3, 6, 2, "affine")                                    # lexicographic: two slabs of 3 layers
    b = sharded.partition_bounds(m.E, 2)
    gids = [m.gid[b[r]:b[r + 1]] for r in range(2)]
    cands, flagged = sharded.local_gathers(m.N, gids, [m.dirichlet[b[r]:b[r + 1]] for r in range(2)])
    plans = [sharded.interface_plan(r, cands) for r in range(2)]
    assert np.array_equal(plans[0][1], plans[1][0]) and plans[0][1].size == (3 * 2 + 1) ** 2
    perm, n_iface = sharded.interface_first(gids[0], plans[0])
    assert n_iface == 9 and sorted(perm[:9].tolist()) == list(range(18, 27)) and perm[9:].tolist() == list(range(18))
    for r in range(2):
        sharded.check_mask_agreement(r, plans[r], flagged)
    broken = [flagged[0], flagged[1][~np.isin(flagged[1], plans[0][1])]]         # rank 1 forgets the shared boundary nodes
    with pytest.raises(ValueError):
        sharded.check_mask_agreement(0, plans[0], broken)
    perm0, n0 = sharded.interface_first(gids[0], {})
    assert n0 == 0 and perm0.tolist() == list(range(27))


def test_partition_rcb():
    sys.path.insert(0, ROOT)
    from paper_2110_01716_b200 import inputs, sharded
    m = inputs.box_mesh(6, 4, 4, 2, "random", seed=1, permute_seed=9)              # scrambled order
    for world in (1, 2, 3, 4, 8):
        parts = sharded.partition_rcb(m.vert, world)
        assert len(parts) == world and sorted(np.concatenate(parts).tolist()) == list(range(m.E))
        sizes = [len(q) for q in parts]
        assert max(sizes) - min(sizes) <= 1 and all(np.all(np.diff(q) > 0) for q in parts)
    parts = sharded.partition_rcb(m.vert, 2)                                        # the longest extent (x) is cut once
    cx = m.vert.reshape(m.E, 8, 3).mean(axis=1)[:, 0]
    assert cx[parts[0]].max() < cx[parts[1]].min()
    cands = [sharded.surface_gids(m.gid[q], m.N) for q in parts]
    assert sharded.interface_plan(0, cands)[1].size == (4 * 2 + 1) ** 2              # one 4 x 4 element plane of nodes

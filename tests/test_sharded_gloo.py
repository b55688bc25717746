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

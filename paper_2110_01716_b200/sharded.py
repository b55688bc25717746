"""NEXT-4: the operator w = M QQ^T (D^T G D + lambda B) u with the ELEMENTS partitioned over ranks,
one process and one GPU per rank (the paper's parallel model: "exchange-and-sum of shared interface
values"; "the user simply provides a global ID for each vertex").

Every step that touches field data runs in the library's kernels (sem_ax_gs, sem_iface_pack, sem_iface_add through the
C ABI); this module only resolves WHICH nodes two ranks share (integer work on the global ids, once, at setup) and moves
the packed buffers between ranks (torch.distributed send/recv over NCCL/NVLink, or an in-process loop-back used by the
one-GPU emulation test).  There is no CPU fallback for the compute: the gloo test of this module drives the same plan
and exchange code with host buffers and checks it against the oracle.

Per application and rank:
    local   w = sem_ax_gs(u)                    (sums the copies inside the rank, applies the mask)
    pack    buf_r[q] = w[first copy of shared node q]            for every rank r that shares nodes with this one
    exchange buf_r <-> rank r                   (pairwise; a node shared by k ranks is exchanged between all pairs)
    add     w[every copy of shared node q] += buf_from_r[q]      in ascending rank order
so that every copy on every rank holds the sum over all ranks.  Interior nodes of a rank are bit-identical to the
single-GPU result; interface nodes agree to round-off (the order of the partial sums differs).
"""
from __future__ import annotations

import numpy as np


def partition_bounds(E: int, world: int):
    """Contiguous element blocks: rank r owns elements [b[r], b[r+1])."""
    return [r * E // world for r in range(world + 1)]


def surface_gids(gid: np.ndarray, N: int) -> np.ndarray:
    """Sorted distinct global ids of the nodes on element surfaces (only these can be shared with another element, hence
    with another rank).  gid: [E, p^3] (or [E, p, p, p]) int64."""
    p = N + 1
    g = np.asarray(gid, dtype=np.int64).reshape(-1, p, p, p)
    on = np.zeros((p, p, p), dtype=bool)
    on[0], on[-1] = True, True
    on[:, 0], on[:, -1] = True, True
    on[:, :, 0], on[:, :, -1] = True, True
    return np.unique(g[:, on])


def interface_plan(rank: int, candidates) -> dict:
    """candidates[r] = surface_gids of rank r (sorted, distinct).  Returns {r: sorted global ids shared with rank r} for
    every other rank that shares at least one node with `rank`.  Both sides compute the same list in the same order."""
    mine = candidates[rank]
    plan = {}
    for r, other in enumerate(candidates):
        if r == rank:
            continue
        shared = np.intersect1d(mine, other, assume_unique=True)
        if shared.size:
            plan[r] = shared
    return plan


class DistComm:
    """torch.distributed plumbing (NCCL on GPUs, gloo on CPU): object all-gather at setup, pairwise send/recv per apply."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)

    def all_gather_arrays(self, a: np.ndarray):
        out = [None] * self.world
        self.dist.all_gather_object(out, a, group=self.group)
        return out

    def exchange(self, send: dict, recv: dict):
        ops = []
        for r in sorted(send):
            ops.append(self.dist.P2POp(self.dist.isend, send[r], r, self.group))
            ops.append(self.dist.P2POp(self.dist.irecv, recv[r], r, self.group))
        if ops:
            for w in self.dist.batch_isend_irecv(ops):
                w.wait()


class ShardedSem:
    """One rank's share of the mesh: a Sem context over its elements plus the interface lists."""

    def __init__(self, comm, E_local, N, vert, gid, dirichlet=None, dtype=None):
        import torch

        from . import binding
        self.comm, self.N = comm, N
        self.sem = binding.Sem(E_local, N, vert, gid, dirichlet)
        self.nL = self.sem.nL
        cand = comm.all_gather_arrays(surface_gids(gid, N))
        self.plan = interface_plan(comm.rank, cand)
        uniq_gid = self.sem.maps()["uniq_gid"]
        self.uniq = {}
        for r, shared in self.plan.items():
            pos = np.searchsorted(uniq_gid, shared)
            assert np.array_equal(uniq_gid[pos], shared)
            self.uniq[r] = torch.from_numpy(pos.astype(np.int32)).cuda()
        self.dtype = dtype or torch.float64
        self.send = {r: torch.empty(u.numel(), device="cuda", dtype=self.dtype) for r, u in self.uniq.items()}
        self.recv = {r: torch.empty_like(b) for r, b in self.send.items()}

    def geom(self, **kw):
        self.sem.geom(**kw)
        return self

    # the three phases, separately callable (the one-GPU emulation interleaves the ranks by hand)
    def local_apply_and_pack(self, u, w, lam: float = 0.0):
        self.sem.ax_gs(u, w, lam)
        self.pack(w)

    def pack(self, w):
        for r in sorted(self.uniq):
            self.sem.iface_pack(self.uniq[r], w, self.send[r])

    def add_received(self, w):
        for r in sorted(self.uniq):                      # ascending rank order on every rank
            self.sem.iface_add(self.uniq[r], self.recv[r], w)

    def gs_across(self, w):
        """The cross-rank part of QQ^T on a field whose copies are already summed inside the rank."""
        self.pack(w)
        self.comm.exchange(self.send, self.recv)
        self.add_received(w)
        return w

    def ax_gs(self, u, w, lam: float = 0.0):
        self.sem.ax_gs(u, w, lam)
        return self.gs_across(w)

    def interface_bytes(self) -> int:
        return sum(int(b.numel()) * b.element_size() for b in self.send.values())

    def close(self):
        self.sem.close()


class LocalComm:
    """In-process stand-in for the setup collectives when several ranks' contexts live in one process on one GPU (the
    emulation the profiling guide asks for when there are fewer GPUs than ranks): all ranks' candidate lists are known."""

    def __init__(self, rank: int, world: int, all_candidates):
        self.rank, self.world, self._cand = rank, world, all_candidates

    def all_gather_arrays(self, a):
        assert np.array_equal(a, self._cand[self.rank])
        return self._cand

    def exchange(self, send, recv):
        raise RuntimeError("LocalComm has no peers: use emulated_ax_gs")


def emulated_ax_gs(shards, us, ws, lam: float = 0.0):
    """All ranks of a partition on ONE GPU, phase by phase: local apply + pack on every rank, buffer hand-over by
    device-to-device copies, add on every rank.  No rank waits on another inside a kernel."""
    for s, u, w in zip(shards, us, ws):
        s.local_apply_and_pack(u, w, lam)
    for a, s in enumerate(shards):
        for r in s.uniq:
            shards[r].recv[a].copy_(s.send[r])
    for s, w in zip(shards, ws):
        s.add_received(w)
    return ws

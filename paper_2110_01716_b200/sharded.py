"""NEXT-4: the operator w = M QQ^T (D^T G D + lambda B) u and the Jacobi-PCG solve with the ELEMENTS
partitioned over ranks, one process and one GPU per rank (the paper's parallel model: "exchange-
and-sum of shared interface values"; "the user simply provides a global ID for each vertex").

Every step that touches field data runs in the library's kernels (sem_ax_gs_sharded, sem_pcg_sharded, sem_iface_pack,
sem_iface_add through the C ABI); this module only resolves WHICH nodes two ranks share (integer work on the global ids,
once, at setup), orders a rank's elements interface-first, and moves the packed buffers and the dot-product scalars
between ranks (torch.distributed over NCCL/NVLink; an in-process stand-in used by the one-GPU emulation tests).  There
is no CPU fallback for the compute: the gloo test of this module drives the same plan and exchange code with host
buffers and checks it against the oracle.

Per application and rank (sem_ax_gs_sharded calls the hooks built here):
    chunk 0   operator + rank-local gather-scatter on the elements that touch shared nodes (they come first)
    gs_begin  buf_r[q] = w[first copy of shared node q] for every peer r; start send/recv with every peer
    the rest  operator + rank-local gather-scatter on the interior elements      (overlaps the exchange)
    gs_end    wait; w[every copy of shared node q] += buf_from_r[q]               in ascending rank order
so that every copy on every rank holds the sum over all ranks.  Nodes of one rank only are bit-identical to the
single-GPU result as long as their copies are summed in the same order (1 or 2 copies: always; more: when the element
order is kept, reorder=False); all other nodes agree to round-off.  A node shared by k ranks is exchanged between all
pairs.
"""
from __future__ import annotations

import threading

import numpy as np


def partition_bounds(E: int, world: int):
    """Contiguous element blocks: rank r owns elements [b[r], b[r+1])."""
    return [r * E // world for r in range(world + 1)]


def partition_rcb(vert: np.ndarray, world: int):
    """Recursive coordinate bisection of the element centroids (vert: [E, 8, 3]): a list of `world` ascending index
    arrays of near-equal size, each a compact box-like piece whatever the element order (the paper partitions with
    parRSB, P:121 -- out of scope; contiguous blocks of a scrambled order would put every element on the interface)."""
    cen = np.asarray(vert, dtype=np.float64).reshape(len(vert), 8, 3).mean(axis=1)

    def split(idx, k):
        if k == 1:
            return [np.sort(idx)]
        kl = k // 2
        ext = cen[idx].max(axis=0) - cen[idx].min(axis=0)
        order = idx[np.argsort(cen[idx, int(np.argmax(ext))], kind="stable")]
        cut = len(idx) * kl // k
        return split(order[:cut], kl) + split(order[cut:], k - kl)

    return split(np.arange(len(cen)), world)


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


def interface_first(gid: np.ndarray, plan: dict):
    """Order of a rank's elements with those touching a shared node first (stable inside both classes).
    Returns (perm, n_iface): new position q holds old element perm[q]."""
    g = np.asarray(gid, dtype=np.int64).reshape(len(gid), -1)
    if not plan:
        return np.arange(len(g)), 0
    shared = np.unique(np.concatenate(list(plan.values())))
    touches = np.isin(g, shared).any(axis=1)
    perm = np.argsort(~touches, kind="stable")
    return perm, int(touches.sum())


def check_mask_agreement(rank: int, plan: dict, flagged):
    """flagged[r] = sorted global ids rank r marks Dirichlet.  A shared node must be marked on both sides or on neither
    (sem.h: "Dirichlet flags must agree between the ranks on shared nodes")."""
    for r, shared in plan.items():
        a, b = np.isin(shared, flagged[rank]), np.isin(shared, flagged[r])
        if not np.array_equal(a, b):
            raise ValueError(f"rank {rank}: {int((a != b).sum())} nodes shared with rank {r} are Dirichlet on one side only")


class _DevView:
    """A raw device address as something torch.as_tensor can wrap without copying."""

    def __init__(self, ptr: int, n: int, typestr: str = "<f8"):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": typestr, "data": (ptr, False), "version": 3}


def device_view(ptr: int, n: int):
    import torch
    return torch.as_tensor(_DevView(ptr, n), device="cuda")


class DistComm:
    """torch.distributed plumbing (NCCL on GPUs, gloo on CPU): object all-gather at setup; per apply pairwise
    send/recv started in one group and waited for later; all-reduce of device scalars."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)

    def all_gather_arrays(self, a: np.ndarray):
        out = [None] * self.world
        self.dist.all_gather_object(out, a, group=self.group)
        return out

    def start_exchange(self, send: dict, recv: dict):
        ops = []
        for r in sorted(send):
            ops.append(self.dist.P2POp(self.dist.isend, send[r], r, self.group))
            ops.append(self.dist.P2POp(self.dist.irecv, recv[r], r, self.group))
        return self.dist.batch_isend_irecv(ops) if ops else []

    def finish_exchange(self, handle):
        for w in handle:
            w.wait()

    def exchange(self, send: dict, recv: dict):
        self.finish_exchange(self.start_exchange(send, recv))

    def allreduce(self, t):
        if self.world > 1:
            self.dist.all_reduce(t, group=self.group)
        return t


class ShardedSem:
    """One rank's share of the mesh: a Sem context over its elements (interface elements first), the interface lists
    and the hooks the library's sharded calls use.  Fields passed to ax_gs / pcg are in the context's element order:
    `to_local(f)` brings a field given in the caller's order of this rank's elements into it, `from_local` back."""

    def __init__(self, comm, E_local, N, vert, gid, dirichlet=None, dtype=None, reorder: bool = True, stream=None):
        import torch

        from . import binding
        self.comm, self.N, self.E = comm, N, E_local
        p3 = (N + 1) ** 3
        gid = np.asarray(gid, dtype=np.int64).reshape(E_local, p3)
        vert = np.asarray(vert, dtype=np.float64).reshape(E_local, 8, 3)
        dirichlet = None if dirichlet is None else np.asarray(dirichlet).reshape(E_local, p3)
        cand = comm.all_gather_arrays(surface_gids(gid, N))
        self.plan = interface_plan(comm.rank, cand)
        flagged = comm.all_gather_arrays(np.unique(gid[dirichlet != 0]) if dirichlet is not None
                                         else np.empty(0, dtype=np.int64))
        check_mask_agreement(comm.rank, self.plan, flagged)
        self.perm, self.n_iface = interface_first(gid, self.plan) if reorder else (np.arange(E_local), 0)
        P = self.perm
        self.sem = binding.Sem(E_local, N, vert[P], gid[P], None if dirichlet is None else dirichlet[P], stream=stream)
        self.stream = self.sem._stream
        self.nL = self.sem.nL
        if reorder and 0 < self.n_iface < E_local:
            self.sem.shard_set_interface(self.n_iface)
        uniq_gid = self.sem.maps()["uniq_gid"]
        self.uniq = {}
        for r, shared in self.plan.items():
            pos = np.searchsorted(uniq_gid, shared)
            assert np.array_equal(uniq_gid[pos], shared)
            self.uniq[r] = torch.from_numpy(pos.astype(np.int32)).cuda()
        self.dtype = dtype or torch.float64
        self._bufs = {}
        self.send, self.recv = self._buffers(self.dtype)
        self._scal = torch.zeros(4, device="cuda", dtype=torch.float64)
        self._pending = None
        self.hooks = binding.ShardHooks(self._gs_begin, self._gs_end, self._allreduce)
        self._prec_dtype = {binding.SEM_F64: torch.float64, binding.SEM_F32: torch.float32}

    # ---- layout ----
    def to_local(self, f):
        """A field over this rank's elements in the caller's order ([E, p^3] or flat, numpy or torch) -> context order."""
        g = f.reshape(self.E, -1)[self.perm if isinstance(f, np.ndarray) else self._perm_t(f)]
        return g.reshape(f.shape)

    def from_local(self, f):
        inv = np.empty_like(self.perm)
        inv[self.perm] = np.arange(self.E)
        g = f.reshape(self.E, -1)[inv if isinstance(f, np.ndarray) else self._perm_t(f, inv)]
        return g.reshape(f.shape)

    def _perm_t(self, f, perm=None):
        import torch
        return torch.from_numpy(np.ascontiguousarray(self.perm if perm is None else perm)).to(f.device)

    def _buffers(self, dtype):
        import torch
        if dtype not in self._bufs:
            send = {r: torch.empty(u.numel(), device="cuda", dtype=dtype) for r, u in self.uniq.items()}
            self._bufs[dtype] = (send, {r: torch.empty_like(b) for r, b in send.items()})
        return self._bufs[dtype]

    def geom(self, **kw):
        self.sem.geom(**kw)
        return self

    # ---- the hooks (called from inside sem_ax_gs_sharded / sem_pcg_sharded, on the calling thread) ----
    def _gs_begin(self, w_ptr: int, prec: int):
        import torch
        send, recv = self._buffers(self._prec_dtype[prec])
        with torch.cuda.stream(self.stream):
            for r in sorted(self.uniq):
                self.sem.iface_pack(self.uniq[r], w_ptr, send[r], prec)
            self._pending = (self.comm.start_exchange(send, recv), recv)

    def _gs_end(self, w_ptr: int, prec: int):
        import torch
        handle, recv = self._pending
        self._pending = None
        with torch.cuda.stream(self.stream):
            self.comm.finish_exchange(handle)
            for r in sorted(self.uniq):                  # ascending rank order on every rank
                self.sem.iface_add(self.uniq[r], recv[r], w_ptr, prec)

    def _allreduce(self, ptr: int, n: int):
        import torch
        with torch.cuda.stream(self.stream):
            self.comm.allreduce(device_view(ptr, n))

    # ---- the sharded calls ----
    def ax_gs(self, u, w, lam: float = 0.0):
        return self.sem.ax_gs_sharded(u, w, self.hooks, lam)

    def pcg(self, b, x, tol: float, maxit: int):
        return self.sem.pcg_sharded(b, x, tol, maxit, self.hooks)

    # ---- the phases, separately callable (the phase-by-phase one-GPU emulation and the CPU tests) ----
    def local_apply_and_pack(self, u, w, lam: float = 0.0):
        self.sem.ax_gs(u, w, lam)
        self.pack(w)

    def pack(self, w):
        for r in sorted(self.uniq):
            self.sem.iface_pack(self.uniq[r], w, self.send[r])

    def add_received(self, w):
        for r in sorted(self.uniq):
            self.sem.iface_add(self.uniq[r], self.recv[r], w)

    def gs_across(self, w):
        """The cross-rank part of QQ^T on a field whose copies are already summed inside the rank."""
        self.pack(w)
        self.comm.exchange(self.send, self.recv)
        self.add_received(w)
        return w

    def interface_bytes(self) -> int:
        return sum(int(b.numel()) * b.element_size() for b in self.send.values())

    def close(self):
        self.sem.close()


class LocalComm:
    """In-process stand-in for the setup collectives when several ranks' contexts live in one process on one GPU (the
    emulation the profiling guide asks for when there are fewer GPUs than ranks): all ranks' lists are known up front.
    `gathers` = the per-rank arrays of every all-gather ShardedSem performs, in order."""

    def __init__(self, rank: int, world: int, *gathers):
        self.rank, self.world, self._gathers, self._k = rank, world, list(gathers), 0

    def all_gather_arrays(self, a):
        g = self._gathers[self._k]
        self._k += 1
        assert np.array_equal(a, g[self.rank])
        return g

    def start_exchange(self, send, recv):
        raise RuntimeError("LocalComm has no peers: use emulated_ax_gs or ThreadComm")

    exchange = start_exchange


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


def local_gathers(N: int, gids, dirichlets):
    """The two all-gathers of ShardedSem's setup for ranks living in one process: (candidates, flagged), one entry per
    rank.  gids[r]: [E_r, p^3] global ids, dirichlets[r]: flags or None."""
    cands = [surface_gids(g, N) for g in gids]
    flagged = [np.unique(np.asarray(g).reshape(len(g), -1)[np.asarray(d).reshape(len(g), -1) != 0]) if d is not None
               else np.empty(0, dtype=np.int64) for g, d in zip(gids, dirichlets)]
    return cands, flagged


class ThreadWorld:
    """State shared by the ThreadComm of every emulated rank (one Python thread per rank, ONE GPU, ONE stream)."""

    def __init__(self, world: int, timeout: float = 120.0):
        import torch
        self.world = world
        self.barrier = threading.Barrier(world, timeout=timeout)
        self.send = [None] * world                      # send[r] = rank r's {peer: buffer} of the exchange in flight
        self.scal = torch.zeros(world, 8, device="cuda", dtype=torch.float64)
        self.stream = None


class ThreadComm(LocalComm):
    """Transport of the one-GPU emulation of sem_ax_gs_sharded / sem_pcg_sharded: every rank runs its library call on its
    own host thread; buffers change hands by device-to-device copies and the all-reduce is a sum over a [world, n]
    device array in a fixed order.  All ranks enqueue on the same stream, so the device executes in the order the host
    threads enqueue, and host barriers (never a kernel) order the threads: pack | barrier | copy | barrier."""

    def __init__(self, tw: ThreadWorld, rank: int, *gathers):
        super().__init__(rank, tw.world, *gathers)
        self.tw = tw

    def start_exchange(self, send, recv):
        self.tw.send[self.rank] = send
        return (send, recv)

    def finish_exchange(self, handle):
        send, recv = handle
        self.tw.barrier.wait()                          # every rank has enqueued its pack kernels
        for r in sorted(recv):
            recv[r].copy_(self.tw.send[r][self.rank])
        self.tw.barrier.wait()                          # every copy is enqueued: the send buffers may be reused

    def exchange(self, send, recv):
        self.finish_exchange(self.start_exchange(send, recv))

    def allreduce(self, t):
        n = t.numel()
        self.tw.scal[self.rank, :n].copy_(t)
        self.tw.barrier.wait()
        t.copy_(self.tw.scal[:, :n].sum(dim=0))
        self.tw.barrier.wait()
        return t


def run_ranks(world: int, fn, tw: ThreadWorld | None = None):
    """fn(rank) on one host thread per rank; returns the results in rank order, re-raises the first failure (and breaks
    the barrier so that the other threads do not wait for a rank that died)."""
    out, err = [None] * world, [None] * world

    def body(r):
        try:
            out[r] = fn(r)
        except BaseException as exc:
            err[r] = exc
            if tw is not None:
                tw.barrier.abort()

    threads = [threading.Thread(target=body, args=(r,)) for r in range(world)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    for e in err:
        if e is not None and not isinstance(e, threading.BrokenBarrierError):
            raise e
    for e in err:
        if e is not None:
            raise e
    return out

"""One grid on several GPUs as x1 slabs (include/hamr.h "x1 slabs over peer memory").

Plumbing only: which process holds which slab, how a neighbour's arena becomes a device pointer in this process (CUDA IPC
through torch's shared CUDA storages, or torch's symmetric memory), and the two ordering points + one MAX reduction per step
(torch.distributed).  Every number of the path is computed by the kernels behind the C-ABI: a slab's ghost fill reads its
neighbours' zones through those pointers (over NVLink between GPUs); nothing is packed, sent or received here.

    partition_x1(n1, parts)            contiguous, balanced x1 ranges (optionally by a per-plane cost)
    Slab                               one hamr_shard_create_in grid (a hamr.Grid: the usual getters work per slab)
    LocalRing                          all slabs in THIS process on one device, stepped in lockstep (tests, 1-GPU measurements)
    DistSlab                           this rank's slab of a torch.distributed job, one process per GPU

PAPER.md:111 (NVLink for intra-node GPU-GPU communication), PAPER.md:93 fn. 2 (one Courant step for the whole grid),
PAPER.md:135, 145 (contiguous runs of the block curve, balanced by cost).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import hamr

NG = 3


def partition_x1(n1: int, parts: int, cost=None):
    """[(i_lo, n1_local)] * parts: contiguous x1 ranges covering [0, n1), each >= 3 zones thick.  cost: per-plane cost
    (length n1; default uniform): range r ends where the running cost first reaches (r + 1) / parts of the total — the
    1-D form of cutting the block curve into runs of equal cost."""
    n1, parts = int(n1), int(parts)
    if parts < 1 or n1 < NG * parts:
        raise ValueError(f"{n1} x1 zones cannot be cut into {parts} slabs of >= {NG}")
    w = np.ones(n1) if cost is None else np.asarray(cost, dtype=np.float64)
    if w.shape != (n1,) or not np.all(w > 0):
        raise ValueError("cost must be n1 positive numbers")
    cum = np.concatenate([[0.0], np.cumsum(w)])
    cuts = [0]
    for r in range(1, parts):
        c = int(np.searchsorted(cum, cum[-1] * r / parts, side="left"))
        if c > 0 and abs(cum[c - 1] - cum[-1] * r / parts) <= abs(cum[c] - cum[-1] * r / parts):
            c -= 1   # the nearer of the two planes around the target
        c = max(c, cuts[-1] + NG)                  # this slab is thick enough
        c = min(c, n1 - NG * (parts - r))          # ... and so can every later one be
        cuts.append(c)
    cuts.append(n1)
    return [(cuts[r], cuts[r + 1] - cuts[r]) for r in range(parts)]


def neighbours(r: int, parts: int, periodic: bool):
    """(low, high) slab index of slab r's x1 neighbours, None at a physical boundary"""
    if parts == 1:
        return None, None
    lo = r - 1 if r > 0 else (parts - 1 if periodic else None)
    hi = r + 1 if r < parts - 1 else (0 if periodic else None)
    return lo, hi


class Slab(hamr.Grid):
    """Zones [i_lo, i_lo + n1) of the grid `p` describes (hamr_shard_create_in).  arena: a torch CUDA uint8 tensor that
    holds the slab (allocated here if None; it is what a neighbour attaches to)."""

    def __init__(self, p: dict, i_lo: int, n1: int, arena=None):
        import torch
        self.L = hamr.lib()
        self.pg = p
        self.i_lo, self.n1 = int(i_lo), int(n1)
        self.p = dict(p, n=(self.n1, int(p["n"][1]), int(p["n"][2])))
        self.n = tuple(self.p["n"])
        self._par = hamr.pack_params(p)
        nbytes = C.c_size_t(0)
        rc = self.L.hamr_shard_workspace_bytes(C.byref(self._par), self.i_lo, self.n1, C.byref(nbytes))
        if rc != hamr.OK:
            raise hamr.HamrError(rc, "hamr_shard_workspace_bytes")
        self.nbytes = nbytes.value
        if arena is None:
            arena = torch.empty(self.nbytes + 256, dtype=torch.uint8, device="cuda")
        self._arena = arena
        self.arena_offset = (-arena.data_ptr()) % 256          # the grid starts at the first 256-byte boundary
        if arena.numel() < self.nbytes + self.arena_offset:
            raise ValueError("arena too small")
        h = C.c_void_p(None)
        rc = self.L.hamr_shard_create_in(C.byref(self._par), self.i_lo, self.n1,
                                         C.c_void_p(arena.data_ptr() + self.arena_offset), C.c_size_t(self.nbytes),
                                         C.c_void_p(torch.cuda.current_stream().cuda_stream), C.byref(h))
        if rc != hamr.OK or not h.value:
            raise hamr.HamrError(rc, "hamr_shard_create_in")
        self.h = h

    @property
    def arena_ptr(self):
        return self._arena.data_ptr() + self.arena_offset

    def attach(self, side, peer_arena_ptr, peer_i_lo, peer_n1):
        self._ck(self.L.hamr_shard_attach(self.h, int(side), C.c_void_p(int(peer_arena_ptr)), int(peer_i_lo), int(peer_n1)))

    def shard_commit(self):
        self._ck(self.L.hamr_shard_commit(self.h))

    def stage(self, k):
        self._ck(self.L.hamr_shard_stage(self.h, int(k)))

    def ctop_get(self, t):
        self._ck(self.L.hamr_shard_ctop_get_dev(self.h, C.c_void_p(t.data_ptr())))

    def ctop_set(self, t):
        self._ck(self.L.hamr_shard_ctop_set_dev(self.h, C.c_void_p(t.data_ptr())))

    def local(self, a, stag=-1):
        """this slab's part of a global dense array (zones, or faces along `stag`)"""
        return np.ascontiguousarray(a[self.i_lo:self.i_lo + self.n1 + (1 if stag == 0 else 0)])


class LocalRing:
    """Every slab of the grid in this process, on the current device and stream, stepped in lockstep.  The kernels and the
    neighbour reads are those of the multi-GPU job (the neighbour's arena is a pointer on the same device); stream order
    stands in for the two ordering points and an elementwise max for the reduction."""

    def __init__(self, p: dict, parts, cost=None):
        import torch
        ranges = partition_x1(p["n"][0], parts, cost) if isinstance(parts, int) else list(parts)
        self.p, self.ranges = p, ranges
        self.slabs = [Slab(p, lo, n) for lo, n in ranges]
        periodic = int(p["bc_lo"][0]) == 0
        for r, s in enumerate(self.slabs):
            for side, q in enumerate(neighbours(r, len(ranges), periodic)):
                if q is not None:
                    s.attach(side, self.slabs[q].arena_ptr, *ranges[q])
        self._ct = torch.zeros((len(ranges), 3), dtype=torch.float64, device="cuda")
        self._mx = torch.zeros(3, dtype=torch.float64, device="cuda")

    def _reduce(self):
        import torch
        for r, s in enumerate(self.slabs):
            s.ctop_get(self._ct[r])
        torch.amax(self._ct, dim=0, out=self._mx)     # the reduction a job does with all_reduce(MAX)
        for s in self.slabs:
            s.ctop_set(self._mx)

    def set_prims(self, hydro, bface=None):
        for s in self.slabs:
            rc = s.set_prims([s.local(h) for h in hydro],
                             None if bface is None else [s.local(b, d) for d, b in enumerate(bface)])
            if rc != hamr.OK:
                return rc
        for s in self.slabs:
            s.shard_commit()
        self._reduce()
        return hamr.OK

    def step_async(self, nsteps=1):
        for _ in range(nsteps):
            for s in self.slabs:
                s.stage(0)
            for s in self.slabs:
                s.stage(1)
            self._reduce()

    def step(self, nsteps=1):
        self.step_async(nsteps)
        for s in self.slabs:
            s.sync()
        return self.slabs[0].t, None

    def get_prims(self):
        parts = [s.get_prims() for s in self.slabs]
        return [np.concatenate([q[c] for q in parts], axis=0) for c in range(8)]

    def get_bface(self):
        parts = [s.get_bface() for s in self.slabs]
        out = []
        for d in range(3):   # the interface face of two slabs is held by both: keep the low slab's up to its last face
            out.append(np.concatenate([q[d][:-1] if (d == 0 and r < len(parts) - 1) else q[d]
                                       for r, q in enumerate(parts)], axis=0))
        return out

    def divb(self):
        return max(s.divb() for s in self.slabs)

    def stats(self):
        return tuple(int(v) for v in np.sum([s.stats() for s in self.slabs], axis=0))

    def launch_count(self):
        return sum(s.launch_count() for s in self.slabs)

    @property
    def t(self):
        return self.slabs[0].t

    @property
    def dt(self):
        return self.slabs[0].dt

    def close(self):
        for s in self.slabs:
            s.close()


class Reducer:
    """MAX over the ranks of a torch.distributed group, in place, on a small tensor — the one reduction of the path (the
    Courant maxima, PAPER.md:93 fn. 2) and, with a dummy tensor, its ordering points.  Backend nccl: an all_reduce on
    the current stream (orders the ranks' streams, does not block the host).  Any other backend: a device tensor goes
    through host memory (the copy synchronises the stream: every kernel enqueued before it has finished on return)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.on_stream = dist.get_backend(group) == "nccl"

    def max_(self, t):
        if self.on_stream or not t.is_cuda:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX, group=self.group)
            return t
        h = t.cpu()
        self.dist.all_reduce(h, op=self.dist.ReduceOp.MAX, group=self.group)
        t.copy_(h)
        return t


class DistSlab:
    """This rank's slab of a torch.distributed job (one process per GPU; torch.cuda.set_device before).
    peer_memory = "ipc": every rank shares its arena as a CUDA IPC handle (torch's shared CUDA storage, gathered with
    all_gather_object) and opens its neighbours'; "symm": the arenas are one torch symmetric-memory allocation
    (rendezvous gives every rank's buffer pointer).  Either way the neighbour's arena is a device pointer this rank's
    ghost kernel dereferences: NVLink / NVSwitch between GPUs.
    Backend nccl: the reductions are all_reduce calls on the grid's (= torch's current) stream, which also order the
    slabs; nothing blocks the host.  Any other backend (gloo: CPU tests, several processes on one GPU): the stream is
    synchronised and three doubles go through host memory."""

    def __init__(self, p: dict, group=None, peer_memory="ipc", cost=None):
        import torch
        import torch.distributed as dist
        self.red = Reducer(group)
        self.dist, self.group = dist, group
        self.rank, self.world = self.red.rank, self.red.world
        self.p = p
        self.ranges = partition_x1(p["n"][0], self.world, cost)
        lo, n1 = self.ranges[self.rank]
        periodic = int(p["bc_lo"][0]) == 0
        nb = neighbours(self.rank, self.world, periodic)
        self._keep = []
        if peer_memory == "symm":
            import torch.distributed._symmetric_memory as symm
            par = hamr.pack_params(p)
            need = 0
            for a, b in self.ranges:    # one size for all ranks
                nbytes = C.c_size_t(0)
                rc = hamr.lib().hamr_shard_workspace_bytes(C.byref(par), a, b, C.byref(nbytes))
                if rc != hamr.OK:
                    raise hamr.HamrError(rc, "hamr_shard_workspace_bytes")
                need = max(need, nbytes.value)
            arena = symm.empty(need + 256, dtype=torch.uint8, device=torch.device("cuda", torch.cuda.current_device()))
            hdl = symm.rendezvous(arena, group if group is not None else dist.group.WORLD)
            self.slab = Slab(p, lo, n1, arena=arena)
            ptrs = [int(v) for v in hdl.buffer_ptrs]
            self._keep.append(hdl)
            peer_ptr = {q: ptrs[q] + ((-ptrs[q]) % 256) for q in nb if q is not None}
        elif peer_memory == "ipc":
            from torch.multiprocessing.reductions import reduce_tensor
            self.slab = Slab(p, lo, n1)
            mine = reduce_tensor(self.slab._arena)
            every = [None] * self.world
            dist.all_gather_object(every, mine, group=group)
            peer_ptr = {}
            for q in set(v for v in nb if v is not None):
                fn, args = every[q]
                t = fn(*args)                       # a tensor over the neighbour's arena (cudaIpcOpenMemHandle)
                self._keep.append(t)
                peer_ptr[q] = t.data_ptr() + ((-t.data_ptr()) % 256)
        else:
            raise ValueError("peer_memory is 'ipc' or 'symm'")
        for side, q in enumerate(nb):
            if q is not None:
                self.slab.attach(side, peer_ptr[q], *self.ranges[q])
        self._ct = torch.zeros(3, dtype=torch.float64, device="cuda")
        self._fence = torch.zeros(1, dtype=torch.float64, device="cuda")

    def _allreduce_max(self, t):
        self.red.max_(t)

    def _reduce(self):
        self.slab.ctop_get(self._ct)
        self._allreduce_max(self._ct)
        self.slab.ctop_set(self._ct)

    def set_prims(self, hydro, bface=None):
        """hydro / bface: the GLOBAL dense arrays (each rank takes its part) — or use self.slab.set_prims with local ones
        followed by commit()"""
        s = self.slab
        rc = s.set_prims([s.local(h) for h in hydro], None if bface is None else [s.local(b, d) for d, b in enumerate(bface)])
        if rc != hamr.OK:
            return rc
        self.commit()
        return hamr.OK

    def commit(self):
        self._allreduce_max(self._fence)             # every slab holds its state
        self.slab.shard_commit()
        self._reduce()

    def step_async(self, nsteps=1):
        for _ in range(nsteps):
            self.slab.stage(0)
            self._allreduce_max(self._fence)         # every slab has finished its predictor
            self.slab.stage(1)
            self._reduce()                           # ... and its corrector: clock, next dt

    def step(self, nsteps=1):
        self.step_async(nsteps)
        self.slab.sync()
        return self.slab.t, None

    def close(self):
        import torch
        torch.cuda.synchronize()
        self.dist.barrier(group=self.group)          # no neighbour reads this arena any more
        self.slab.close()
        self._keep.clear()

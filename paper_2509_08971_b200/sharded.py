"""NEXT-4 (SURVEY §8(e),(f)): z-slab sharding of one simulation over several GPUs, one process per GPU.

Each rank owns a contiguous slab of z-planes in its own `Hard` context.  Before each RK stage the g boundary
planes of every field travel to the neighbouring ranks (NCCL send/recv of two packed device buffers per
direction, 96 MB per face per stage at 896^2 x g = 3: ~0.1 ms over NVLink against an ~80 ms stage), and once per
step the max wavespeed is all-reduced (MAX) in place in the device scalar block, so every rank derives the
same dt on the device: nothing returns to the host inside a step.  All arithmetic stays in the CUDA kernels;
this module only sequences `hard_substep` phases and the exchanges.

Communicators with one interface: `DistComm` (torch.distributed on the tensors as they are: NCCL with device
buffers on GPUs, gloo with host tensors in the CPU tests of the exchange logic), `HostStagedComm` (the same pairing
code, device buffers staged through pinned host memory — for a backend that cannot move device memory, i.e. gloo:
this is how the real `ShardedHard` class is exercised with several processes sharing ONE GPU, where NCCL cannot
run), and `LocalGroup` (several ranks emulated by one process on one GPU: the phases of all ranks run in lockstep
and halos are copied directly).  In none of them does a kernel wait on another rank.
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import hard

PH_GHOST_U, PH_STAGE1, PH_GHOST_U1, PH_STAGE2, PH_END = range(5)


def split_z(nz, world):
    """Contiguous z ranges [k0, k1) of the `world` slabs (sizes differ by at most one plane)."""
    base, rem = divmod(nz, world)
    out, k = [], 0
    for r in range(world):
        n = base + (1 if r < rem else 0)
        out.append((k, k + n))
        k += n
    return out


def neighbours(rank, world, periodic):
    """(lower, upper) neighbour ranks of `rank`, None at a physical boundary."""
    lo = rank - 1 if rank > 0 else (world - 1 if periodic else None)
    hi = rank + 1 if rank < world - 1 else (0 if periodic else None)
    return lo, hi


class DistComm:
    """Halo exchange and max-reduction over torch.distributed (one process per rank)."""

    def __init__(self, periodic):
        import torch.distributed as dist
        self.dist = dist
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        self.lo, self.hi = neighbours(self.rank, self.world, periodic)

    def exchange(self, send_low, send_high, recv_low, recv_high):
        """send_low goes to the lower neighbour (it arrives in its recv_high), send_high to the upper one."""
        dist = self.dist
        if self.world == 1:                                  # periodic wrap onto oneself
            if self.lo is not None:
                recv_low.copy_(send_high)
                recv_high.copy_(send_low)
            return
        ops = []
        if self.lo is not None:
            ops.append(dist.P2POp(dist.isend, send_low, self.lo))
            ops.append(dist.P2POp(dist.irecv, recv_low, self.lo))
        if self.hi is not None:
            ops.append(dist.P2POp(dist.isend, send_high, self.hi))
            ops.append(dist.P2POp(dist.irecv, recv_high, self.hi))
        if self.world == 2 and self.lo is not None and self.lo == self.hi:
            # two ranks, periodic: both faces go to the same peer; order the pairs so that they match
            ops = [dist.P2POp(dist.isend, send_low, self.lo), dist.P2POp(dist.isend, send_high, self.hi),
                   dist.P2POp(dist.irecv, recv_high, self.hi), dist.P2POp(dist.irecv, recv_low, self.lo)]
        for req in dist.batch_isend_irecv(ops):
            req.wait()

    def allreduce_max(self, t):
        if self.world > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)


class HostStagedComm(DistComm):
    """DistComm for a backend that only moves host memory (gloo): the four halo buffers and the lambda slot are
    staged through pinned host tensors around the very same send/recv pairing and all-reduce.  The staging copies
    run on the current CUDA stream, which is synchronised before the host-side exchange and implicitly ordered
    after it (the copy back is enqueued on the same stream), so the kernels see the halos they would with NCCL."""

    def __init__(self, periodic):
        super().__init__(periodic)
        self._host = {}

    def _pinned(self, key, like):
        import torch
        t = self._host.get(key)
        if t is None or t.numel() != like.numel():
            t = torch.empty(like.numel(), dtype=like.dtype, pin_memory=True)
            self._host[key] = t
        return t

    def exchange(self, send_low, send_high, recv_low, recv_high):
        import torch
        dev = (send_low, send_high, recv_low, recv_high)
        host = [self._pinned(k, t) for k, t in zip(("sl", "sh", "rl", "rh"), dev)]
        host[0].copy_(send_low, non_blocking=True)
        host[1].copy_(send_high, non_blocking=True)
        torch.cuda.current_stream().synchronize()
        super().exchange(*host)
        if self.lo is not None:
            recv_low.copy_(host[2], non_blocking=True)
        if self.hi is not None:
            recv_high.copy_(host[3], non_blocking=True)

    def allreduce_max(self, t):
        import torch
        if self.world > 1:
            h = self._pinned("lam", t)
            h.copy_(t, non_blocking=True)
            torch.cuda.current_stream().synchronize()
            super().allreduce_max(h)
            t.copy_(h, non_blocking=True)


class Slab:
    """One rank's slab: a `Hard` context over (nx, ny, nz_local) plus its halo buffers."""

    def __init__(self, n, gamma, bc, rank, world, scheme=hard.SCHEME_WENO5Z_HLL, spacing=None, radiation=False):
        import torch
        self.torch = torch
        nx, ny, nz = n
        self.rank, self.world = rank, world
        self.k0, self.k1 = split_z(nz, world)[rank]
        self.lo, self.hi = neighbours(rank, world, bc == hard.BC_PERIODIC)
        sp = spacing if spacing is not None else (1.0 / nx, 1.0 / ny, 1.0 / nz)
        self.h = hard.Hard(nx, ny, self.k1 - self.k0, gamma, bc, scheme=scheme, spacing=sp, radiation=radiation)
        self.h.set_slab(self.lo is not None, self.hi is not None)
        m = self.h.halo_doubles()
        mk = lambda: torch.empty(m, dtype=torch.float64, device="cuda")
        self.send_low, self.send_high, self.recv_low, self.recv_high = mk(), mk(), mk(), mk()

    def set_state(self, fields):
        """fields: the five global arrays (nz, ny, nx) or this rank's slab of them."""
        loc = [f[self.k0:self.k1] if f.shape[0] != self.k1 - self.k0 else f for f in fields]
        loc = [np.ascontiguousarray(a) if isinstance(a, np.ndarray) else a.contiguous() for a in loc]
        self.h.set_state(*loc)

    def lam_tensor(self, nxt):
        """The lambda slot of the device scalar block as a 1-element float64 tensor (no copy)."""
        torch = self.torch
        ptr = self.h.lambda_ptr(nxt)
        ws = self.h.ws
        off = ptr - ws.data_ptr()
        return ws[off:off + 8].view(torch.float64)

    def pack(self, buffer):
        if self.lo is not None:
            self.h.halo_pack(buffer, 0, self.send_low)
        if self.hi is not None:
            self.h.halo_pack(buffer, 1, self.send_high)

    def unpack(self, buffer):
        if self.lo is not None:
            self.h.halo_unpack(buffer, 0, self.recv_low)
        if self.hi is not None:
            self.h.halo_unpack(buffer, 1, self.recv_high)

    def get_state(self):
        return self.h.get_state()

    def close(self):
        self.h.close()


class ShardedHard:
    """One rank of a sharded run (use under torchrun, one process per GPU)."""

    def __init__(self, n, gamma, bc, scheme=hard.SCHEME_WENO5Z_HLL, spacing=None, radiation=False, comm=None):
        if comm is None:                       # NCCL moves device buffers itself; gloo needs the host staging
            import torch.distributed as dist
            # a group initialised without an explicit backend reports a composite string ("cuda:nccl,cpu:gloo")
            use_nccl = "nccl" in str(dist.get_backend()).lower()
            comm = (DistComm if use_nccl else HostStagedComm)(bc == hard.BC_PERIODIC)
            if comm.rank == 0:
                import sys
                print("ShardedHard: %s (backend %s)" % (type(comm).__name__, dist.get_backend()), file=sys.stderr)
        self.comm = comm
        self.slab = Slab(n, gamma, bc, self.comm.rank, self.comm.world, scheme, spacing, radiation)

    def set_state(self, fields):
        self.slab.set_state(fields)
        self.comm.allreduce_max(self.slab.lam_tensor(0))

    def _exchange(self, buffer):
        s = self.slab
        s.pack(buffer)
        self.comm.exchange(s.send_low, s.send_high, s.recv_low, s.recv_high)
        s.unpack(buffer)

    def step(self, cfl, nsteps=1):
        s = self.slab
        for _ in range(nsteps):
            self._exchange(0)
            s.h.substep(PH_GHOST_U, cfl=cfl)
            s.h.substep(PH_STAGE1, cfl=cfl)
            self._exchange(1)
            s.h.substep(PH_GHOST_U1, cfl=cfl)
            s.h.substep(PH_STAGE2, cfl=cfl)
            self.comm.allreduce_max(s.lam_tensor(1))
            s.h.substep(PH_END, cfl=cfl)

    def get_state(self):
        return self.slab.get_state()

    def max_dt(self):
        return self.slab.h.max_dt()

    def close(self):
        self.slab.close()


class LocalGroup:
    """All ranks of a sharded run emulated in ONE process on one GPU, phases in lockstep (tests)."""

    def __init__(self, n, gamma, bc, world, scheme=hard.SCHEME_WENO5Z_HLL, spacing=None, radiation=False):
        self.slabs = [Slab(n, gamma, bc, r, world, scheme, spacing, radiation) for r in range(world)]
        self.world = world

    def _allreduce(self, nxt):
        import torch
        ts = [s.lam_tensor(nxt) for s in self.slabs]
        m = torch.stack(ts).max(dim=0).values
        for t in ts:
            t.copy_(m)

    def _exchange(self, buffer):
        for s in self.slabs:
            s.pack(buffer)
        for s in self.slabs:                      # what DistComm.exchange does with send/recv
            if s.lo is not None:
                s.recv_low.copy_(self.slabs[s.lo].send_high)
            if s.hi is not None:
                s.recv_high.copy_(self.slabs[s.hi].send_low)
        for s in self.slabs:
            s.unpack(buffer)

    def set_state(self, fields):
        for s in self.slabs:
            s.set_state(fields)
        self._allreduce(0)

    def step(self, cfl, nsteps=1):
        for _ in range(nsteps):
            self._exchange(0)
            for ph in (PH_GHOST_U, PH_STAGE1):
                for s in self.slabs:
                    s.h.substep(ph, cfl=cfl)
            self._exchange(1)
            for ph in (PH_GHOST_U1, PH_STAGE2):
                for s in self.slabs:
                    s.h.substep(ph, cfl=cfl)
            self._allreduce(1)
            for s in self.slabs:
                s.h.substep(PH_END, cfl=cfl)

    def get_state(self):
        parts = [s.get_state() for s in self.slabs]
        return [np.concatenate([p[f] for p in parts], axis=0) for f in range(5)]

    def max_dt(self):
        return self.slabs[0].h.max_dt()

    def close(self):
        for s in self.slabs:
            s.close()

"""NEXT-4 (sec.9 "parallelisation to multiple GPUs per host"): the smear step and the
plaquette on a lattice decomposed along t.

Rank r of R owns the time slices [r*Lt, (r+1)*Lt), Lt = L3/R, and keeps them in a LOCAL lattice of t-extent Lt + 2:
local slice 0 is the halo from rank r-1 (its last own slice), slices 1..Lt are the rank's own, slice Lt+1 is the halo
from rank r+1 (its first own slice); periodic in t over the ranks.  Every operand of the staple sum of an own site lies
in the local lattice: the diagonal neighbour x - t^ + mu^ (mu spatial) is inside the received slice, so a 1-d split
needs no corner exchange.  Per step and neighbour one time slice of the four link fields moves (31.9 MB at 48^3x96
fp32 with two ranks); a slice is one contiguous range of a field's storage (lqx_field_slice).

One smear step:   1. post the halo exchange of the input links (side stream / non-blocking requests),
                  2. launch the INTERIOR own slices [2, Lt) -- they read no halo --,
                  3. wait for the halos, launch the two boundary slices [1, 2) and [Lt, Lt+1).
The plaquette of the own sites reads slice Lt+1 too, then one all-reduce of a double.

This module is plumbing: WHO exchanges WHAT and WHICH slices a launch covers.  The arithmetic is behind a `backend`
(`LqxBackend`: the CUDA library through its C-ABI; the tests also drive it with the CPU oracle to check the
partition logic without a GPU) and the transport behind a `comm` (`DistComm`: torch.distributed, NCCL on GPUs / gloo on
CPU; `SelfComm`: one rank, the halos are the rank's own periodic images; the tests add an in-process emulation of
several ranks).  BASELINE.json's contract stays "replicas only" (`bench.py --gpus N`); this is the widening of SURVEY 8(f).
"""
from __future__ import annotations


def local_dims(global_dims, world):
    L0, L1, L2, L3 = (int(d) for d in global_dims)
    if L3 % world:
        raise ValueError(f"L3 = {L3} is not a multiple of {world} ranks")
    if L3 // world < 2:
        raise ValueError("every rank needs at least two own time slices")
    return (L0, L1, L2, L3 // world + 2)


def own_range(global_dims, rank, world):
    lt = int(global_dims[3]) // world
    return rank * lt, (rank + 1) * lt


class SelfComm:
    """One rank: the neighbour in both directions is the rank itself."""
    rank, world = 0, 1

    def exchange(self, send_lo, send_hi, recv_lo, recv_hi):
        """recv_lo <- previous rank's send_hi, recv_hi <- next rank's send_lo.  Returns a handle for wait()."""
        for dst, src in zip(recv_lo, send_hi):
            dst.copy_(src)
        for dst, src in zip(recv_hi, send_lo):
            dst.copy_(src)
        return None

    def wait(self, handle):
        pass

    def allreduce_sum(self, x: float) -> float:
        return x


class DistComm:
    """torch.distributed point-to-point on the default group: NCCL for CUDA tensors, gloo for CPU tensors."""

    def __init__(self):
        import torch.distributed as dist

        self.dist = dist
        self.rank, self.world = dist.get_rank(), dist.get_world_size()

    def exchange(self, send_lo, send_hi, recv_lo, recv_hi):
        dist = self.dist
        prev, nxt = (self.rank - 1) % self.world, (self.rank + 1) % self.world
        ops = []
        for k, t in enumerate(send_lo):  # my first own slice -> the previous rank's upper halo
            ops.append(dist.P2POp(dist.isend, t, prev, tag=2 * k))
        for k, t in enumerate(send_hi):  # my last own slice -> the next rank's lower halo
            ops.append(dist.P2POp(dist.isend, t, nxt, tag=2 * k + 1))
        for k, t in enumerate(recv_hi):
            ops.append(dist.P2POp(dist.irecv, t, nxt, tag=2 * k))
        for k, t in enumerate(recv_lo):
            ops.append(dist.P2POp(dist.irecv, t, prev, tag=2 * k + 1))
        return dist.batch_isend_irecv(ops)

    def wait(self, handle):
        for req in handle or []:
            req.wait()

    def allreduce_sum(self, x: float) -> float:
        import torch

        t = torch.tensor([x], dtype=torch.float64)
        if self.dist.get_backend() == "nccl":
            t = t.cuda()
        self.dist.all_reduce(t)
        return float(t.item())


class LqxBackend:
    """The CUDA library on a rank's local lattice (fields = lqx Field objects with torch-owned memory)."""

    def __init__(self, lqx, lat):
        self.lqx, self.lat = lqx, lat

    def slice(self, field, t):
        return field.slice_view(t)

    def smear_range(self, uout, uin, alpha, t0, t1):
        self.lqx.smear_step_range(uout, uin, alpha, t0, t1)

    def plaquette_range(self, u, t0, t1):
        return self.lqx.plaquette_range(u, t0, t1)

    def side_stream(self):
        import torch

        return torch.cuda.Stream(device=self.lat.device)


class TSplit:
    """The driver of one rank.  `lt` own slices in a local lattice of t-extent lt + 2."""

    def __init__(self, backend, comm, global_dims):
        self.be, self.comm = backend, comm
        self.global_dims = tuple(int(d) for d in global_dims)
        self.dims = local_dims(global_dims, comm.world)
        self.lt = self.dims[3] - 2

    def _halo_views(self, u):
        be, lt = self.be, self.lt
        send_lo = [be.slice(f, 1) for f in u]        # first own slice
        send_hi = [be.slice(f, lt) for f in u]       # last own slice
        recv_lo = [be.slice(f, 0) for f in u]        # halo below
        recv_hi = [be.slice(f, lt + 1) for f in u]   # halo above
        return send_lo, send_hi, recv_lo, recv_hi

    def exchange_halos(self, u):
        h = self.comm.exchange(*self._halo_views(u))
        self.comm.wait(h)

    def smear_step(self, uout, uin, alpha, overlap=True, halos_fresh=False):
        """uout's own slices <- one smear step of uin (own slices + fresh halos).  uout's halo slices are NOT valid
        afterwards: the next step exchanges them.  halos_fresh: the caller has exchanged uin's halos already."""
        lt = self.lt
        if halos_fresh:
            self.be.smear_range(uout, uin, alpha, 1, lt + 1)
        elif overlap and lt > 2:
            h = self.comm.exchange(*self._halo_views(uin))
            self.be.smear_range(uout, uin, alpha, 2, lt)          # interior: needs slices 1 .. lt only
            self.comm.wait(h)
            self.be.smear_range(uout, uin, alpha, 1, 2)
            self.be.smear_range(uout, uin, alpha, lt, lt + 1)
        else:
            self.exchange_halos(uin)
            self.be.smear_range(uout, uin, alpha, 1, lt + 1)

    def plaquette_sum(self, u, halos_fresh=False):
        """Global plaquette sum: the own sites of every rank (they read the upper halo), all-reduced."""
        if not halos_fresh:
            self.exchange_halos(u)
        return self.comm.allreduce_sum(self.be.plaquette_range(u, 1, self.lt + 1))

    def smear_iterate(self, u, tmp, alpha, nsteps):
        """nsteps steps in place on ping-pong fields; returns the global plaquette average after each step."""
        vol = 1
        for d in self.global_dims:
            vol *= d
        plaqs = []
        cur, nxt = u, tmp
        for _ in range(nsteps):
            self.smear_step(nxt, cur, alpha)
            cur, nxt = nxt, cur
            plaqs.append(self.plaquette_sum(cur) / (18.0 * vol))
        return cur, plaqs

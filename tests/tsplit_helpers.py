"""Test-side pieces of the NEXT-4 t-split (paper_1105_2279_b200/tsplit.py): a backend that does the arithmetic with
the CPU ORACLE on a rank's local lattice (so the partition / halo / slice logic can be checked without a GPU), the
scatter / gather between a global field and the ranks' local fields, and an in-process emulation of R ranks."""
import numpy as np
import torch

import oracle as orc


def v3_of(dims):
    return int(dims[0]) * int(dims[1]) * int(dims[2])


def scatter(global_field, global_dims, rank, world):
    """rank's local field [(lt+2)*V3, ...]: own slices in 1..lt, halos filled with the periodic neighbours' slices."""
    v3, lt = v3_of(global_dims), int(global_dims[3]) // world
    g = np.asarray(global_field).reshape((int(global_dims[3]), v3) + global_field.shape[1:])
    t0 = rank * lt
    idx = [(t0 - 1) % global_dims[3]] + list(range(t0, t0 + lt)) + [(t0 + lt) % global_dims[3]]
    return np.ascontiguousarray(g[idx].reshape((-1,) + global_field.shape[1:]))


def scatter_no_halo(global_field, global_dims, rank, world):
    """the same with the halo slices poisoned: they must come from the exchange"""
    loc = scatter(global_field, global_dims, rank, world)
    v3 = v3_of(global_dims)
    loc[:v3] = np.nan
    loc[-v3:] = np.nan
    return loc


def gather_own(local_fields_by_rank, global_dims):
    """concatenate the ranks' own slices -> global field"""
    v3 = v3_of(global_dims)
    return np.concatenate([np.asarray(f)[v3:-v3] for f in local_fields_by_rank], axis=0)


class OracleBackend:
    """fields: torch CPU tensors [Vloc, 3, 3, 2] (a time slice is rows [t*V3, (t+1)*V3)); arithmetic by the oracle on
    the local lattice, of which only the requested slices are kept"""

    def __init__(self, local_dims, variant):
        self.dims, self.variant, self.v3 = tuple(local_dims), variant, v3_of(local_dims)

    def slice(self, field, t):
        return field[t * self.v3:(t + 1) * self.v3]

    def smear_range(self, uout, uin, alpha, t0, t1):
        full = orc.smear_step(self.dims, [f.numpy() for f in uin], alpha, self.variant)
        for o, f in zip(uout, full):
            o[t0 * self.v3:t1 * self.v3] = torch.from_numpy(f[t0 * self.v3:t1 * self.v3])

    def plaquette_range(self, u, t0, t1):
        sites = np.arange(t0 * self.v3, t1 * self.v3, dtype=np.int64)
        return float(orc.plaquette_sites(self.dims, [f.numpy() for f in u], sites, self.variant).sum())


class EmulatedRanks:
    """R ranks in one process, run one after the other: comm objects whose exchange() only records what a rank
    sends and receives; `flush()` then moves the data between the ranks' buffers (any tensor type with copy_)."""

    def __init__(self, world):
        self.world = world
        self.pending = {}

    def comm(self, rank):
        outer = self

        class _Comm:
            def __init__(self):
                self.rank, self.world = rank, outer.world
                self.partial = None

            def exchange(self, send_lo, send_hi, recv_lo, recv_hi):
                outer.pending[rank] = (send_lo, send_hi, recv_lo, recv_hi)
                return None

            def wait(self, handle):
                pass

            def allreduce_sum(self, x):
                self.partial = x
                return x

        return _Comm()

    def flush(self):
        for r, (_, _, recv_lo, recv_hi) in self.pending.items():
            prev, nxt = (r - 1) % self.world, (r + 1) % self.world
            for dst, src in zip(recv_lo, self.pending[prev][1]):  # previous rank's last own slice
                dst.copy_(src)
            for dst, src in zip(recv_hi, self.pending[nxt][0]):   # next rank's first own slice
                dst.copy_(src)
        self.pending = {}

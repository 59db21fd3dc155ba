"""Time-slab domain decomposition of the D_w apply over ranks (first step).

The paper's codes run on rank-local lattices with a neighbour map between ranks and exchange
boundary data before the operator is applied.  Here the lattice is cut along time, T_loc = T / world
slices per rank.  Every rank works on a LOCAL lattice of T_loc + 2 slices: its own slices plus one ghost slice below
and one above.  Gauge field and U(1) field of the ghost slices are part of the rank's fields (loaded once); the ghost
slices of the spinor are filled by one exchange with the two time neighbours before every apply (torch.distributed
send/recv: NCCL over NVLink between GPUs, gloo in the CPU tests).  The existing single-GPU kernels then run unchanged
on the local lattice and the ghost slices of the result are discarded: every interior site sees exactly the neighbours,
links and clover leaves of the global lattice (a leaf reaches one site from its corner), so the decomposition is correct
by construction.  The local lattice is periodic in its own time direction, which only couples the two ghost slices to
each other; the global antiperiodic boundary condition is carried by the sign of the time links of global slice T-1
(reading R9), which cancels in every clover leaf.  C* boundaries are spatial and stay rank-local.

This module is host logic only (index arithmetic, slicing, the exchange).  What applies the operator is passed in: the
CUDA context on a GPU rank, the oracle in the CPU tests.  Cost of this first step: 2 / T_loc redundant work and one
exchange per apply that is not yet overlapped with the interior; both are what a fused halo kernel would remove.
"""
from __future__ import annotations

import numpy as np


class TimeSlabs:
    """Geometry of rank `rank` of `world` for a global physical lattice dims = (T, L1, L2, L3)."""

    def __init__(self, dims, world: int, rank: int):
        T = int(dims[0])
        if world < 1 or not (0 <= rank < world):
            raise ValueError("TimeSlabs: need world >= 1 and 0 <= rank < world")
        if T % world or (T // world) % 2 or T // world < 2:
            raise ValueError("TimeSlabs: T must split into an even number (>= 2) of slices per rank")
        self.dims = tuple(int(d) for d in dims)
        self.world, self.rank = world, rank
        self.T, self.T_loc = T, T // world
        self.t0 = rank * self.T_loc
        self.local_dims = (self.T_loc + 2,) + self.dims[1:]
        self.prev, self.next = (rank - 1) % world, (rank + 1) % world

    def time_index(self):
        """Global time slice of every local slice (ghost below, interior, ghost above)."""
        return [(self.t0 - 1 + k) % self.T for k in range(self.T_loc + 2)]

    def local_fields(self, U, A=None, antiperiodic=True):
        """Rank-local gauge field (and U(1) field) including the ghost slices.  With antiperiodic fermions the time links
        of global slice T-1 carry the factor -1 and the local context is created WITHOUT the antiperiodic bit."""
        idx = self.time_index()
        Ul = np.ascontiguousarray(np.asarray(U)[idx])
        if antiperiodic:
            for k, t in enumerate(idx):
                if t == self.T - 1:
                    Ul[k, ..., 0, :, :] *= -1.0
        Al = None if A is None else np.ascontiguousarray(np.asarray(A)[idx])
        return Ul, Al

    @staticmethod
    def local_bc(cstar: int) -> int:
        """bc word of the local context: same C* directions, periodic in (local) time."""
        return int(cstar) & 3

    def scatter(self, psi_global):
        """Interior slices of this rank from a global extended-lattice spinor [T][X1][L2][L3][4][3], with empty ghosts."""
        psi_global = np.asarray(psi_global)
        loc = np.zeros((self.T_loc + 2,) + psi_global.shape[1:], dtype=psi_global.dtype)
        loc[1:self.T_loc + 1] = psi_global[self.t0:self.t0 + self.T_loc]
        return loc

    def interior(self, local):
        return local[1:self.T_loc + 1]


def exchange_time_ghosts(ts: TimeSlabs, local, dist=None):
    """Fill the two ghost slices of `local` (tensor or array [T_loc+2][...]) from the time neighbours.  world == 1:
    periodic self-copy.  The four point-to-point operations go out as ONE batch (dist.batch_isend_irecv = one
    ncclGroupStart/End under NCCL): NCCL ignores tags and serialises the p2p operations of a peer pair on one stream, so
    with world == 2 (previous and next rank are the same peer) four separately issued isend/irecv calls could block each
    other; inside a group they cannot.  The pairing does not rely on tags: for every peer both sides list the upward
    message (my last interior slice -> the next rank's lower ghost) before the downward one, and messages between a pair
    of ranks are matched in issue order."""
    Tl = ts.T_loc
    if ts.world == 1 or dist is None:
        if ts.world != 1:
            raise ValueError("exchange_time_ghosts: a process group is needed for world > 1")
        local[0] = local[Tl]
        local[Tl + 1] = local[1]
        return local
    import torch
    t = local if isinstance(local, torch.Tensor) else torch.from_numpy(local)
    up_send, down_send = t[Tl].contiguous(), t[1].contiguous()
    low_recv, high_recv = torch.empty_like(up_send), torch.empty_like(down_send)
    ops = [dist.P2POp(dist.isend, up_send, ts.next), dist.P2POp(dist.irecv, low_recv, ts.prev),       # upward
           dist.P2POp(dist.isend, down_send, ts.prev), dist.P2POp(dist.irecv, high_recv, ts.next)]    # downward
    for r in dist.batch_isend_irecv(ops):
        r.wait()
    t[0].copy_(low_recv)
    t[Tl + 1].copy_(high_recv)
    return local


def apply_Dw_distributed(ts: TimeSlabs, local_psi, apply_local, dist=None):
    """One distributed D_w apply: exchange the ghost slices, apply the local operator `apply_local(local_psi) -> local_out`
    (the CUDA context of this rank, or the oracle in CPU tests) on the T_loc + 2 lattice, return the interior slices."""
    exchange_time_ghosts(ts, local_psi, dist)
    out = apply_local(local_psi)
    return ts.interior(out.reshape(local_psi.shape))

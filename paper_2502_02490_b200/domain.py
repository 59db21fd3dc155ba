"""Domain decomposition of the D_w apply and solve over ranks.

The paper's codes run on rank-local lattices, exchange boundary data before the operator is applied
 and realise C* boundary conditions by changing the neighbour map between ranks ("shifted boundaries",
PAPER.md:137-139).  Here:

* :class:`ProcessGrid` is that neighbour map as a pure function: a hop across the global boundary of a C* direction
  k in 2..cstar lands, on the lattice doubled in direction 1, displaced by L1 in direction 1 -- on the rank N1/2 further
  along direction 1 if that direction is distributed, else on the same rank column with a LOCAL displacement by L1.
* :class:`LocalLattice` is a rank's lattice: its own sites plus ghost layers in the cut directions, any of the four (time: one tile = 4 slices
  thick, so that the owned sites are whole time slabs of the device site order and nothing is computed on ghosts; directions
  2 and 3: two layers, the one next to the owned sites carrying data).  Gauge and U(1) fields of the ghost layers are loaded with the rank's fields, once.
* :func:`halo_exchange` fills the spinor ghost layers: the boundary layer is spin-projected to 12 reals per site by a kernel
  (qxd_face_gather), the face buffers travel as ONE batch of point-to-point operations (NCCL between GPUs), and
  qxd_face_scatter writes the ghost spinors, displaced by L1 where the message crossed a C* boundary.
* :class:`GpuRank` applies D_w and the even-odd operator D-hat with the unchanged single-GPU kernels on the owned time slabs:
  interior slabs are launched first and run while the faces are in flight, the two boundary slabs after the ghosts have arrived.
* :func:`cgne` is the distributed CG on the normal equations: every scalar is all-reduced over the ranks.

The module is written against two small interfaces so that the same code runs (a) one rank per process under
torch.distributed (``TorchComm``; NCCL on GPUs, gloo in the CPU tests) and (b) all ranks of a decomposition inside one
process, one after the other (``LocalComm``: how a decomposition is verified on the single GPU a test box has).  What applies
the operator on a rank is an ``ops`` object: :class:`GpuRank` here, the fp64 oracle in the CPU tests.
"""
from __future__ import annotations

import numpy as np

TIME_GHOST = 4          # thickness of the time ghost zones = tile extent b0 of the device site order
SPACE_GHOST = 2         # thickness of the ghost zones of directions 2 and 3 (keeps the local extent a multiple of the tile extent 4;
                        # only the layer next to the owned sites carries data)


class ProcessGrid:
    """Ranks on a 4D grid, direction 3 fastest; the C* neighbour map of PAPER.md:139 as a pure function."""

    def __init__(self, dims, grid, cstar=0):
        self.dims = tuple(int(d) for d in dims)              # global PHYSICAL extents T, L1, L2, L3
        self.grid = tuple(int(n) for n in grid)
        self.cstar = int(cstar)
        self.ext = (self.dims[0], (2 if cstar else 1) * self.dims[1], self.dims[2], self.dims[3])   # extended lattice
        for mu in range(4):
            if self.grid[mu] < 1 or self.ext[mu] % self.grid[mu] or (self.ext[mu] // self.grid[mu]) % 2:
                raise ValueError("ProcessGrid: every direction must split into an even number of sites per rank")
        if cstar and self.grid[1] > 1 and self.grid[1] % 2:
            raise ValueError("ProcessGrid: with C* boundaries direction 1 (doubled) needs an even number of ranks")
        self.local_ext = tuple(self.ext[mu] // self.grid[mu] for mu in range(4))
        self.world = int(np.prod(self.grid))

    def coords(self, rank):
        c = []
        for n in reversed(self.grid):
            c.append(rank % n)
            rank //= n
        return tuple(reversed(c))

    def rank(self, coords):
        r = 0
        for c, n in zip(coords, self.grid):
            r = r * n + (c % n)
        return r

    def neighbour(self, rank, mu, direction):
        """(rank of the neighbour in direction +-mu, local displacement in direction 1 applied to data that arrive from / go
        to it, crossed): a hop over the global boundary of a C* direction k (2 <= k <= cstar) is displaced by L1 on the doubled
        lattice: N1/2 ranks along direction 1 if it is distributed, else L1 sites locally."""
        c = list(self.coords(rank))
        n = c[mu] + direction
        crossed = n < 0 or n >= self.grid[mu]
        c[mu] = n % self.grid[mu]
        shift1 = 0
        if crossed and 2 <= mu <= self.cstar:
            if self.grid[1] > 1:
                c[1] = (c[1] + self.grid[1] // 2) % self.grid[1]
            else:
                shift1 = self.dims[1]
        return self.rank(c), shift1, crossed

    def owner(self, x):
        """Rank that owns the extended global site x, and its local (ghost-free) coordinates."""
        c = tuple(x[mu] // self.local_ext[mu] for mu in range(4))
        return self.rank(c), tuple(x[mu] % self.local_ext[mu] for mu in range(4))


class LocalLattice:
    """The lattice of one rank: owned sites + ghost layers in the cut directions.

    Directions 0, 2, 3: the rank keeps the whole doubled direction 1 and its context is a C* lattice of its own.  A cut along
    direction 1 (the paper's layout: the mirror half of the doubled lattice lives on OTHER ranks) makes the
    local lattice an ordinary periodic one: direction 1 and every C* direction get ghost zones, the hop across the global
    boundary of a C* direction arrives from the rank N1/2 further along direction 1 (ProcessGrid.neighbour), and the gauge
    field of the sites with extended coordinate x1 >= L1 is the mirror image conj(U), -A."""

    def __init__(self, pg: ProcessGrid, rank: int, antiperiodic=True, force_cut=(False, False, False, False)):
        self.pg, self.rank = pg, rank
        self.c = pg.coords(rank)
        cut = [pg.grid[mu] > 1 or bool(force_cut[mu]) for mu in range(4)]
        if cut[1] and not pg.cstar:
            raise ValueError("LocalLattice: direction 1 is cut only on C* lattices (use directions 0, 2, 3 otherwise)")
        if cut[1]:
            for mu in range(2, pg.cstar + 1):      # their wrap leaves the rank: they need ghost zones whatever grid[mu] is
                cut[mu] = True
        self.cut = tuple(cut)
        self.g = (TIME_GHOST if cut[0] else 0, SPACE_GHOST if cut[1] else 0, SPACE_GHOST if cut[2] else 0, SPACE_GHOST if cut[3] else 0)
        T, L1, L2, L3 = pg.dims
        X1 = (2 if pg.cstar else 1) * L1
        # owned extents: PHYSICAL in the directions of a C* context, EXTENDED in direction 1 when it is cut (the context is then periodic)
        self.own = (T // pg.grid[0], X1 // pg.grid[1] if cut[1] else L1, L2 // pg.grid[2], L3 // pg.grid[3])
        self.local_dims = tuple(self.own[mu] + 2 * self.g[mu] for mu in range(4))
        self.origin = (self.c[0] * self.own[0], self.c[1] * self.own[1] if cut[1] else 0, self.c[2] * self.own[2], self.c[3] * self.own[3])
        # boundary conditions of the local context: a cut direction is handled by the ghosts (periodic locally, which only
        # couples ghost layers to each other).  The library's C* directions are 1..cstar, so the uncut C* directions must
        # still be a prefix: cutting direction 3 drops the count to 2, cutting 2 (and 3, if it is a C* direction) to 1,
        # cutting 1 to 0
        cs = pg.cstar
        if cut[1]:
            cs = 0
        elif cs == 3 and cut[2] and not cut[3]:
            raise ValueError("LocalLattice: with cstar = 3 a cut along direction 2 needs direction 3 cut too (force_cut) -- "
                             "the local C* directions must be 1..k")
        elif cs >= 2 and cut[2]:
            cs = 1
        elif cs == 3 and cut[3]:
            cs = 2
        self.cstar_local = cs
        self.antiperiodic = bool(antiperiodic)
        self.bc_local = self.cstar_local | ((1 if (antiperiodic and not cut[0]) else 0) << 2)
        self.local_ext = (self.local_dims[0], self.local_dims[1] if cut[1] else X1, self.local_dims[2], self.local_dims[3])   # extended local lattice (spinors)
        if cut[0] and (self.own[0] % TIME_GHOST or self.own[0] < 2 * TIME_GHOST):
            raise ValueError("LocalLattice: a time cut needs T_loc to be a multiple of 4 and >= 8 (whole tiles, two boundary slabs)")

    # ---- index maps -------------------------------------------------------------------------------------------------
    def _global_index(self):
        """For every local site of the context's lattice (incl. ghosts): global PHYSICAL coordinates and whether the site is a
        C* mirror image: mirror[x1, y, z] (x1 in the mirror half of the doubled lattice when direction 1 is cut, XOR an odd
        number of C* boundary crossings in directions 2 and 3)."""
        T, L1, L2, L3 = self.pg.dims
        t = (self.origin[0] - self.g[0] + np.arange(self.local_dims[0])) % T
        if self.cut[1]:
            x1e = (self.origin[1] - self.g[1] + np.arange(self.local_dims[1])) % (2 * L1)
            x1, m1 = x1e % L1, x1e >= L1
        else:
            x1, m1 = np.arange(L1), np.zeros(L1, dtype=bool)
        yr = self.origin[2] - self.g[2] + np.arange(self.local_dims[2])
        zr = self.origin[3] - self.g[3] + np.arange(self.local_dims[3])
        y, z = yr % L2, zr % L3
        my = ((yr // L2) % 2 != 0) & (self.pg.cstar >= 2)
        mz = ((zr // L3) % 2 != 0) & (self.pg.cstar == 3)
        return t, x1, y, z, m1[:, None, None] ^ my[None, :, None] ^ mz[None, None, :]

    def local_fields(self, U, A=None):
        """Rank-local gauge field (and U(1) field) including the ghost layers.  With antiperiodic fermions and a time cut the
        time links of global slice T-1 carry the factor -1 (the local context is then periodic in time); links of sites
        that are C* mirror images are conj(U), -A (reading R8)."""
        t, x1, y, z, mirror = self._global_index()
        U = np.asarray(U)
        Ul = np.ascontiguousarray(U[t][:, x1][:, :, y][:, :, :, z])
        Ul[:, mirror] = np.conj(Ul[:, mirror])
        if self.antiperiodic and self.cut[0]:
            Ul[t == self.pg.dims[0] - 1, ..., 0, :, :] *= -1.0
        Al = None
        if A is not None:
            Al = np.ascontiguousarray(np.asarray(A)[t][:, x1][:, :, y][:, :, :, z])
            Al[:, mirror] *= -1.0
        return Ul, Al

    def owned_slices(self):
        return tuple(slice(self.g[mu], self.g[mu] + self.own[mu]) if self.cut[mu] else slice(None) for mu in range(4))

    def _global_slices(self):
        o = self.origin
        return tuple(slice(o[mu], o[mu] + self.own[mu]) if self.cut[mu] else slice(None) for mu in range(4))

    def scatter(self, psi_global):
        """Owned part of a global extended-lattice spinor [T][X1][L2][L3][4][3] placed into a local array with empty ghosts."""
        psi_global = np.asarray(psi_global)
        loc = np.zeros(self.local_ext + psi_global.shape[4:], dtype=psi_global.dtype)
        loc[self.owned_slices()] = psi_global[self._global_slices()]
        return loc

    def gather_into(self, psi_global, local):
        psi_global[self._global_slices()] = np.asarray(local).reshape(self.local_ext + psi_global.shape[4:])[self.owned_slices()]

    def messages(self):
        """The halo messages this rank SENDS, one per cut direction and side: dicts with the layer to gather (coord, sign of
        the projector the receiver's hop applies), the destination rank, the ghost layer it fills there and the displacement
        in direction 1 the receiver applies (C* shifted boundary)."""
        out = []
        for mu in (3, 2, 1, 0):     # the spatial directions first: their ghosts are needed by every time slab
            if not self.cut[mu]:
                continue
            g, n = self.g[mu], self.own[mu]
            up, s_up, _ = self.pg.neighbour(self.rank, mu, +1)
            dn, s_dn, _ = self.pg.neighbour(self.rank, mu, -1)
            # upward: my last owned layer -> lower ghost of the next rank, read there by backward hops: (1 + gamma_mu)
            out.append(dict(mu=mu, side="up", coord=g + n - 1, sign=-1, dst=up, ghost=g - 1, shift1=s_up))
            # downward: my first owned layer -> upper ghost of the previous rank, read there by forward hops: (1 - gamma_mu)
            out.append(dict(mu=mu, side="down", coord=g, sign=+1, dst=dn, ghost=g + n, shift1=s_dn))
        return out


# ---------------------------------------------------------------------------------------------------------------------
# communication: one rank per process (torch.distributed) or all ranks in one process (verification on one device)
# ---------------------------------------------------------------------------------------------------------------------
class LocalComm:
    """All ranks of the decomposition live in this process (ops[r] for every rank r); messages are copies."""

    def __init__(self, world):
        self.world = world
        self.my_ranks = list(range(world))

    def exchange(self, sends):
        """sends: list of (src, dst, tag, tensor).  Returns {(dst, tag): tensor}."""
        return {(dst, tag): t.clone() for (src, dst, tag, t) in sends}

    def allreduce_sum(self, per_rank):
        """per_rank: {rank: 0-d / 1-element tensor}; every tensor is replaced by the sum over ranks, in place."""
        vals = list(per_rank.values())
        tot = vals[0].clone()
        for v in vals[1:]:
            tot += v.to(tot.device)
        for v in vals:
            v.copy_(tot.to(v.device))


class TorchComm:
    """One rank per process under torch.distributed (NCCL on GPUs, gloo on CPU).  All point-to-point operations of an
    exchange go out as ONE batch (one ncclGroup): NCCL ignores tags and serialises the operations of a peer pair on one
    stream, so separately issued sends and receives between two ranks could block each other; messages between a pair are
    matched by issue order, which is the same on both sides (directions 3, 2, 0, upward before downward).  A message to
    the rank itself (a direction with a single rank but ghosts) is a copy unless `self_via_dist` asks for a real send/recv
    pair (how the NCCL path is exercised on a single GPU)."""

    def __init__(self, dist, self_via_dist=False):
        self.dist = dist
        self.world = dist.get_world_size()
        self.rank = dist.get_rank()
        self.my_ranks = [self.rank]
        self.self_via_dist = self_via_dist

    def exchange(self, sends, recv_like):
        """sends: list of (src = me, dst, tag, tensor); recv_like: list of (src, tag, template tensor) in the SAME order in
        which the peers list their sends.  Returns {(me, tag): tensor}."""
        import torch
        dist = self.dist
        out, ops = {}, []
        for (src, dst, tag, t) in sends:
            if dst == self.rank and not self.self_via_dist:
                continue
            ops.append(dist.P2POp(dist.isend, t, dst))
        for (src, tag, like) in recv_like:
            if src == self.rank and not self.self_via_dist:
                mine = [t for (s, d, tg, t) in sends if d == self.rank and tg == tag]
                out[(self.rank, tag)] = mine[0].clone()
                continue
            buf = torch.empty_like(like)
            out[(self.rank, tag)] = buf
            ops.append(dist.P2POp(dist.irecv, buf, src))
        if ops:
            for r in dist.batch_isend_irecv(ops):
                r.wait()
        return out

    def allreduce_sum(self, per_rank):
        for v in per_rank.values():
            if self.world > 1:
                self.dist.all_reduce(v)


def halo_exchange(comm, lats, ops, vecs, parity_mask=3, directions=(3, 2, 1, 0), g5in=False):
    """Fill the ghost layers of the spinors vecs[r] (r over the ranks this process holds) in the given cut directions.
    Gather kernels -> one batched exchange -> scatter kernels.  The tag of a message is (mu, side).  g5in: the operator pass
    applies gamma5 to its input (D-hat^dagger): the ghosts must then hold the projection of gamma5 psi, and since the upper
    components of (1 - s gamma_mu) gamma5 psi are those of (1 + s gamma_mu) psi, the faces are gathered with the opposite sign
    (gamma5 leaves the expanded ghost spinor (h, 0) unchanged)."""
    sends, recv_like = [], {}
    for r in comm.my_ranks:
        for m in lats[r].messages():
            if m["mu"] not in directions:
                continue
            buf = ops[r].face_gather(vecs[r], parity_mask, m["mu"], m["coord"], -m["sign"] if g5in else m["sign"])
            sends.append((r, m["dst"], (m["mu"], m["side"]), buf))
    if isinstance(comm, LocalComm):
        arrived = comm.exchange(sends)
    else:
        r = comm.my_ranks[0]
        rl = []
        for m in lats[r].messages():          # what I receive mirrors what I send: the "up" message comes from below
            if m["mu"] not in directions:
                continue
            src = lats[r].pg.neighbour(r, m["mu"], -1 if m["side"] == "up" else +1)[0]
            like = [t for (s, d, tg, t) in sends if tg == (m["mu"], m["side"])][0]
            rl.append((src, (m["mu"], m["side"]), like))
        arrived = comm.exchange(sends, rl)
    for r in comm.my_ranks:
        lat = lats[r]
        for mu in directions:
            if not lat.cut[mu]:
                continue
            g, n = lat.g[mu], lat.own[mu]
            for side, ghost, d in (("up", g - 1, -1), ("down", g + n, +1)):
                shift1 = lat.pg.neighbour(r, mu, d)[1]      # displacement of data that crossed my lower / upper boundary
                ops[r].face_scatter(vecs[r], parity_mask, mu, ghost, shift1, arrived[(r, (mu, side))])


def halo_clear(lats, ops, vecs, ranks, parity_mask=3):
    """Zero the ghost layers (after the operator has used them), so that reductions over a vector see owned sites only."""
    for r in ranks:
        lat = lats[r]
        for mu in (0, 1, 2, 3):
            if lat.cut[mu]:
                g, n = lat.g[mu], lat.own[mu]
                ops[r].halo_zero(vecs[r], parity_mask, mu, 0, g)
                ops[r].halo_zero(vecs[r], parity_mask, mu, g + n, 2 * g + n)


# ---------------------------------------------------------------------------------------------------------------------
# a rank on a GPU: the C-ABI library on the local lattice
# ---------------------------------------------------------------------------------------------------------------------
class GpuRank:
    """One rank's CUDA context on its local lattice (fields with ghost layers loaded once) and the per-rank steps of the
    distributed operator.  Vectors are packed FULL-lattice buffers of the storage precision `prec` (torch uint8 tensors)."""

    def __init__(self, lat: LocalLattice, U, A, qel, kappa, q, csw, csw_qed, prec=0, device="cuda:0", pairing=None, extra_precisions=()):
        from . import binding as B
        self.B, self.lat, self.prec = B, lat, prec
        Ul, Al = lat.local_fields(U, A)
        self.g = B.Qxd(*lat.local_dims, lat.bc_local, precisions=tuple({B.QXD_F64, prec} | set(extra_precisions)), device=device, pairing=pairing)
        self.g.gauge_load(Ul, Al, qel)
        self.g.set_quark(kappa, q)
        self.g.clover_build(csw, csw_qed)
        self.nslabs, self.thick = self.g.time_slabs()
        gs = lat.g[0] // self.thick
        self.owned = (gs, self.nslabs - gs)                       # owned time slabs [lo, hi)
        self.hb = self.g.packed_spinor_bytes(prec, half_only=True)

    def close(self):
        self.g.close()

    def with_prec(self, prec):
        """The same context seen through another bound storage precision (the sloppy operator of a mixed-precision solve)."""
        import copy
        o = copy.copy(self)
        o.prec = prec
        o.hb = self.g.packed_spinor_bytes(prec, half_only=True)
        return o

    # vectors
    def alloc(self):
        return self.g.new_packed(self.prec)

    def pack(self, local_nat):
        return self.g.spinor_pack(np.ascontiguousarray(local_nat), self.prec)

    def unpack(self, v):
        return self.g.spinor_unpack(v, self.prec).cpu().numpy().reshape(self.lat.local_ext + (4, 3))

    def half(self, v, parity=0):
        return v[parity * self.hb:(parity + 1) * self.hb]

    # halo kernels
    def face_gather(self, v, pmask, mu, coord, sign):
        buf = self.g.face_buffer(self.prec, mu)
        return self.g.face_gather(v, self.prec, pmask, mu, coord, sign, buf)

    def face_scatter(self, v, pmask, mu, coord, shift1, buf):
        self.g.face_scatter(v, self.prec, pmask, mu, coord, shift1, buf)

    def halo_zero(self, v, pmask, mu, lo, hi):
        self.g.halo_zero(v, self.prec, pmask, mu, lo, hi)

    # operator passes on a range of owned time slabs: which = "interior", "boundary" or "all"
    def slab_ranges(self, which):
        lo, hi = self.owned
        if not self.lat.cut[0] or which == "all":
            return [(lo, hi)] if which in ("all", "interior") else []
        return [(lo + 1, hi - 1)] if which == "interior" else [(lo, lo + 1), (hi - 1, hi)]

    def dslash(self, which, mode, vin, vout, parity_out=0, flags=0, phi=None):
        for rng in self.slab_ranges(which):
            if rng[1] > rng[0]:
                self.g.dslash_packed(mode, vin, vout, self.prec, parity_out=parity_out, flags=flags, phi=phi, slabs=rng)


def _pass(comm, lats, ops, vin, vout, mode, flags=0, parity_out=0, phi=None, overlap=True):
    """One dslash-shaped pass of the distributed operator on every rank of this process: ghosts of directions 3 and 2 first (every slab
    needs them), then the time faces -- in flight while the interior slabs run when there is one rank per process."""
    ranks = comm.my_ranks
    pm = 3 if mode == 0 else (1 << (1 - parity_out))
    g5in = bool(flags & 1)        # QXD_DSF_G5IN
    if any(lats[r].cut[1] or lats[r].cut[2] or lats[r].cut[3] for r in ranks):
        halo_exchange(comm, lats, ops, vin, pm, directions=(3, 2, 1), g5in=g5in)
    time_cut = any(lats[r].cut[0] for r in ranks)
    ph = {r: (phi[r] if phi is not None else None) for r in ranks}
    if time_cut and overlap and isinstance(comm, TorchComm) and vin[ranks[0]].is_cuda:
        import torch
        r = ranks[0]
        main = torch.cuda.current_stream()
        if not hasattr(comm, "side"):
            comm.side = torch.cuda.Stream()
        sends = [(r, m["dst"], (m["mu"], m["side"]), ops[r].face_gather(vin[r], pm, m["mu"], m["coord"], -m["sign"] if g5in else m["sign"]))
                 for m in lats[r].messages() if m["mu"] == 0]
        rl = [(lats[r].pg.neighbour(r, 0, -1 if m["side"] == "up" else +1)[0], (0, m["side"]), t)
              for m, (_, _, _, t) in zip([m for m in lats[r].messages() if m["mu"] == 0], sends)]
        e1 = torch.cuda.Event()
        e1.record(main)
        with torch.cuda.stream(comm.side):
            comm.side.wait_event(e1)
            arrived = comm.exchange(sends, rl)
            e2 = torch.cuda.Event()
            e2.record(comm.side)
        ops[r].dslash("interior", mode, vin[r], vout[r], parity_out, flags, ph[r])     # runs while the faces travel
        main.wait_event(e2)
        g, n = lats[r].g[0], lats[r].own[0]
        for side, ghost, d in (("up", g - 1, -1), ("down", g + n, +1)):
            ops[r].face_scatter(vin[r], pm, 0, ghost, lats[r].pg.neighbour(r, 0, d)[1], arrived[(r, (0, side))])
        ops[r].dslash("boundary", mode, vin[r], vout[r], parity_out, flags, ph[r])
    else:
        if time_cut:
            halo_exchange(comm, lats, ops, vin, pm, directions=(0,), g5in=g5in)
        for r in ranks:
            ops[r].dslash("all", mode, vin[r], vout[r], parity_out, flags, ph[r])
    halo_clear(lats, ops, vin, ranks, pm)
    # time ghosts are never computed (whole slabs are skipped); the ghost layers of directions 2 and 3 lie inside the owned slabs and
    # do receive (meaningless) results: clear them, so that the output is zero outside the owned sites
    pmo = 3 if mode == 0 else (1 << parity_out)
    for r in ranks:
        for mu in (1, 2, 3):
            if lats[r].cut[mu]:
                g, n = lats[r].g[mu], lats[r].own[mu]
                ops[r].halo_zero(vout[r], pmo, mu, 0, g)
                ops[r].halo_zero(vout[r], pmo, mu, g + n, 2 * g + n)


class GpuOperator:
    """The distributed operators on GPU ranks: D_w on full-lattice vectors and D-hat = A_ee - D_eo A_oo^{-1} D_oe on the even
    halves (vectors are dicts rank -> packed buffer; the odd half of `tmp` is the intermediate of D-hat)."""

    def __init__(self, comm, lats, ops, overlap=True):
        self.comm, self.lats, self.ops, self.overlap = comm, lats, ops, overlap
        self.ranks = comm.my_ranks
        self.tmp = {r: ops[r].alloc() for r in self.ranks}
        import torch
        self.torch = torch

    def alloc(self):
        return {r: self.ops[r].alloc() for r in self.ranks}

    def apply_Dw(self, vin, vout):
        _pass(self.comm, self.lats, self.ops, vin, vout, 0, overlap=self.overlap)

    def apply(self, vin, vout, dagger=False):
        """vout_e = D-hat vin_e (dagger: D-hat^dagger)."""
        B = self.ops[self.ranks[0]].B
        _pass(self.comm, self.lats, self.ops, vin, self.tmp, B.QXD_DS_HOP_AINV, flags=B.QXD_DSF_G5IN if dagger else 0, parity_out=1, overlap=self.overlap)
        _pass(self.comm, self.lats, self.ops, self.tmp, vout, B.QXD_DS_A_XMHOP, flags=B.QXD_DSF_G5HOP if dagger else 0, parity_out=0, phi=vin,
              overlap=self.overlap)

    # even-odd source preparation and reconstruction (row a8), distributed
    def prepare(self, eta, b):
        """b_e = eta_e - D_eo A_oo^{-1} eta_o"""
        B = self.ops[self.ranks[0]].B
        for r in self.ranks:
            self.ops[r].g.clover_apply_packed(eta[r], self.tmp[r], self.ops[r].prec, 1, inverse=True)
        _pass(self.comm, self.lats, self.ops, self.tmp, b, B.QXD_DS_X_MHOP, parity_out=0, phi=eta, overlap=self.overlap)

    def reconstruct(self, eta, x):
        """x_o = A_oo^{-1}(eta_o - D_oe x_e), written into the odd half of x"""
        B = self.ops[self.ranks[0]].B
        _pass(self.comm, self.lats, self.ops, x, x, B.QXD_DS_AINV_X_MHOP, parity_out=1, phi=eta, overlap=self.overlap)

    # BLAS on the even halves with device-resident, all-reduced scalars
    def scalar(self):
        return {r: self.torch.zeros(1, dtype=self.torch.float64, device=self.ops[r].g.device) for r in self.ranks}

    def norm2(self, v, out):
        for r in self.ranks:
            o = self.ops[r]
            o.g.blas_norm2_dev(o.half(v[r]), o.prec, out[r])
        self.comm.allreduce_sum(out)

    def cg_xr(self, num, den, p, t, x, rvec, rr):
        for r in self.ranks:
            o = self.ops[r]
            o.g.blas_cg_xr(o.prec, num[r], den[r], o.half(p[r]), o.half(t[r]), o.half(x[r]), o.half(rvec[r]), rr[r])
        self.comm.allreduce_sum(rr)

    def cg_p(self, num, den, s, p):
        for r in self.ranks:
            o = self.ops[r]
            o.g.blas_cg_p(o.prec, num[r], den[r], o.half(s[r]), o.half(p[r]))

    def copy(self, x, y):
        for r in self.ranks:
            o = self.ops[r]
            o.g.blas_copy(o.half(x[r]), o.half(y[r]), o.prec)

    def value(self, s):
        return float(s[self.ranks[0]].item())


def cgne(op, b, tol2_abs, maxiter=10000):
    """Distributed CG on the normal equations of `op` keeping the system residual (reading R11), x = 0 start:
    s = A^dag r, p = s, gam = |s|^2; loop: t = A p; al = gam/|t|^2; x += al p; r -= al t; stop on |r|^2 <= tol2_abs;
    s = A^dag r; gam' = |s|^2; p = s + (gam'/gam) p.  Every scalar is a sum over all ranks (all-reduce).  Returns x, info."""
    x, r, s, p, t = op.alloc(), op.alloc(), op.alloc(), op.alloc(), op.alloc()
    gam, gam2, tt, rr = op.scalar(), op.scalar(), op.scalar(), op.scalar()
    op.copy(b, r)
    op.norm2(r, rr)
    it, res2 = 0, op.value(rr)
    if res2 > tol2_abs:
        op.apply(r, s, dagger=True)
        op.copy(s, p)
        op.norm2(s, gam)
    while res2 > tol2_abs and it < maxiter:
        op.apply(p, t)
        op.norm2(t, tt)
        op.cg_xr(gam, tt, p, t, x, r, rr)
        it += 1
        op.apply(r, s, dagger=True)        # enqueued before the host reads |r|^2: the device does not idle on the round trip
        op.norm2(s, gam2)
        res2 = op.value(rr)
        if not (res2 == res2) or res2 <= tol2_abs:
            break
        op.cg_p(gam2, gam, s, p)
        gam, gam2 = gam2, gam
    return x, dict(iters=it, res2=res2, status=0 if res2 <= tol2_abs else -5)


def solve_distributed(op: GpuOperator, eta, tol, maxiter=10000):
    """Solve D_w psi = eta on the decomposed lattice by even-odd preconditioning + distributed CGNE (fp64 storage).
    eta: dict rank -> packed full-lattice buffer with clean ghosts.  Returns psi (same form) and a report."""
    n2 = op.scalar()
    tot = 0.0
    for par in (0, 1):      # |eta|^2 over both parities and all ranks
        for r in op.ranks:
            o = op.ops[r]
            o.g.blas_norm2_dev(o.half(eta[r], par), o.prec, n2[r])
        op.comm.allreduce_sum(n2)
        tot += op.value(n2)
    b = op.alloc()
    op.prepare(eta, b)
    x, info = cgne(op, b, tol * tol * tot, maxiter)
    op.reconstruct(eta, x)
    info["true_res_eo"] = (info["res2"] / tot) ** 0.5 if tot > 0 else 0.0
    return x, info


def solve_distributed_mixed(op_hi: GpuOperator, op_lo: GpuOperator, eta, tol, delta=0.1, maxiter=10000, op_vec: GpuOperator = None):
    """Mixed-precision distributed solve: the CG iteration on the normal equations of D-hat runs on the SLOPPY operator
    op_lo (fp32 storage; same ranks and contexts as op_hi, see GpuRank.with_prec), the solution is accumulated and the true
    residual recomputed with the fp64 operator op_hi whenever the iterated residual has dropped by `delta` since the last
    update ("reliable updates", PAPER.md:207 ref [4]; the single-GPU loop of csrc/solver.cu with every scalar all-reduced and a
    halo exchange inside every operator application).  Convergence is declared on the fp64 residual only.

    op_vec (fp32 view of the same contexts) with a binary16 op_lo: the Krylov vectors x, r, p stay in fp32 and only the operator's
    inputs and outputs (p16, r16, s, t: what travels in the halos) are binary16 -- the form of the single-GPU solver (reading R12;
    rounding x, r, p themselves to binary16 costs 2.8 x the iterations)."""
    if op_vec is not None:
        return _solve_distributed_h16(op_hi, op_lo, op_vec, eta, tol, delta, maxiter)
    H, L = op_hi, op_lo
    ranks = H.ranks
    n2 = H.scalar()
    tot = 0.0
    for par in (0, 1):
        for r in ranks:
            o = H.ops[r]
            o.g.blas_norm2_dev(o.half(eta[r], par), o.prec, n2[r])
        H.comm.allreduce_sum(n2)
        tot += H.value(n2)
    stop2 = tol * tol * tot
    b = H.alloc()
    H.prepare(eta, b)
    xhi, rhi, thi = H.alloc(), H.alloc(), H.alloc()
    xlo, rlo, s, p, t = L.alloc(), L.alloc(), L.alloc(), L.alloc(), L.alloc()
    gam, gam2, tt, rr, rrt = L.scalar(), L.scalar(), L.scalar(), L.scalar(), H.scalar()

    def to_lo(src, dst):
        for r in ranks:
            oh, ol = H.ops[r], L.ops[r]
            oh.g.blas_convert(oh.half(src[r]), oh.prec, ol.half(dst[r]), ol.prec)

    def reliable():
        for r in ranks:
            oh, ol = H.ops[r], L.ops[r]
            oh.g.blas_acc_hi(ol.half(xlo[r]), ol.prec, oh.half(xhi[r]))
        H.apply(xhi, thi)
        for r in ranks:
            oh = H.ops[r]
            oh.g.blas_sub_norm_dev(oh.half(b[r]), oh.half(thi[r]), oh.half(rhi[r]), oh.prec, rrt[r])
        H.comm.allreduce_sum(rrt)
        to_lo(rhi, rlo)
        return H.value(rrt)

    H.copy(b, rhi)
    H.norm2(rhi, rrt)
    rr_true = H.value(rrt)
    to_lo(rhi, rlo)
    it, nrel, maxr = 0, 0, rr_true ** 0.5
    status = 0 if rr_true <= stop2 else -5
    if status:
        L.apply(rlo, s, dagger=True)
        L.copy(s, p)
        L.norm2(s, gam)
    while status and it < maxiter:
        L.apply(p, t)
        L.norm2(t, tt)
        L.cg_xr(gam, tt, p, t, xlo, rlo, rr)
        it += 1
        # s = A^dag r is enqueued BEFORE the host reads |r|^2 (as in csrc/solver.cu): the device never idles on the round trip;
        # the work is only wasted in the iterations that do a reliable update
        L.apply(rlo, s, dagger=True)
        L.norm2(s, gam2)
        res2 = L.value(rr)
        if not (res2 == res2):
            break
        rn = res2 ** 0.5
        maxr = max(maxr, rn)
        if rn < delta * maxr or res2 <= stop2:
            rr_true = reliable()
            nrel += 1
            maxr = rr_true ** 0.5
            if rr_true <= stop2:
                status = 0
                break
            L.apply(rlo, s, dagger=True)
            L.norm2(s, gam2)
        L.cg_p(gam2, gam, s, p)
        gam, gam2 = gam2, gam
    if status:
        rr_true = reliable()
        nrel += 1
        if rr_true <= stop2:
            status = 0
    H.reconstruct(eta, xhi)
    return xhi, dict(iters=it, n_reliable=nrel, status=status, true_res_eo=(rr_true / tot) ** 0.5 if tot > 0 else 0.0)


def _solve_distributed_h16(H: GpuOperator, L: GpuOperator, V: GpuOperator, eta, tol, delta, maxiter):
    """solve_distributed_mixed with a binary16 operator L and fp32 Krylov vectors (allocated through V)."""
    ranks = H.ranks
    n2 = H.scalar()
    tot = 0.0
    for par in (0, 1):
        for r in ranks:
            o = H.ops[r]
            o.g.blas_norm2_dev(o.half(eta[r], par), o.prec, n2[r])
        H.comm.allreduce_sum(n2)
        tot += H.value(n2)
    stop2 = tol * tol * tot
    b = H.alloc()
    H.prepare(eta, b)
    xhi, rhi, thi = H.alloc(), H.alloc(), H.alloc()
    xlo, rlo, p = V.alloc(), V.alloc(), V.alloc()                 # fp32
    r16, p16, s, t = L.alloc(), L.alloc(), L.alloc(), L.alloc()   # binary16
    gam, gam2, tt, rr, rrt = L.scalar(), L.scalar(), L.scalar(), L.scalar(), H.scalar()

    def convert(src, osrc, dst, odst):
        for r in ranks:
            a, c = osrc.ops[r], odst.ops[r]
            a.g.blas_convert(a.half(src[r]), a.prec, c.half(dst[r]), c.prec)

    def reliable():
        for r in ranks:
            oh, ov = H.ops[r], V.ops[r]
            oh.g.blas_acc_hi(ov.half(xlo[r]), ov.prec, oh.half(xhi[r]))
        H.apply(xhi, thi)
        for r in ranks:
            oh = H.ops[r]
            oh.g.blas_sub_norm_dev(oh.half(b[r]), oh.half(thi[r]), oh.half(rhi[r]), oh.prec, rrt[r])
        H.comm.allreduce_sum(rrt)
        convert(rhi, H, rlo, V)
        convert(rhi, H, r16, L)
        return H.value(rrt)

    H.copy(b, rhi)
    H.norm2(rhi, rrt)
    rr_true = H.value(rrt)
    convert(rhi, H, rlo, V)
    convert(rhi, H, r16, L)
    it, nrel, maxr = 0, 0, rr_true ** 0.5
    status = 0 if rr_true <= stop2 else -5
    if status:
        L.apply(r16, s, dagger=True)
        convert(s, L, p, V)
        L.copy(s, p16)
        L.norm2(s, gam)
    while status and it < maxiter:
        L.apply(p16, t)
        L.norm2(t, tt)
        for r in ranks:
            ol, ov = L.ops[r], V.ops[r]
            ol.g.blas_cg_xr_h(gam[r], tt[r], ol.half(p16[r]), ol.half(t[r]), ov.half(xlo[r]), ov.half(rlo[r]), ol.half(r16[r]), rr[r])
        L.comm.allreduce_sum(rr)
        it += 1
        L.apply(r16, s, dagger=True)          # enqueued before the host reads |r|^2 (see solve_distributed_mixed)
        L.norm2(s, gam2)
        res2 = L.value(rr)
        if not (res2 == res2):
            break
        rn = res2 ** 0.5
        maxr = max(maxr, rn)
        if rn < delta * maxr or res2 <= stop2:
            rr_true = reliable()
            nrel += 1
            maxr = rr_true ** 0.5
            if rr_true <= stop2:
                status = 0
                break
            L.apply(r16, s, dagger=True)
            L.norm2(s, gam2)
        for r in ranks:
            ol, ov = L.ops[r], V.ops[r]
            ol.g.blas_cg_p_h(gam2[r], gam[r], ol.half(s[r]), ov.half(p[r]), ol.half(p16[r]))
        gam, gam2 = gam2, gam
    if status:
        rr_true = reliable()
        nrel += 1
        if rr_true <= stop2:
            status = 0
    H.reconstruct(eta, xhi)
    return xhi, dict(iters=it, n_reliable=nrel, status=status, true_res_eo=(rr_true / tot) ** 0.5 if tot > 0 else 0.0)

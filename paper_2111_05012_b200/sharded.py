"""The sharded fine operator: D on a lattice partitioned over ranks (the paper's own runs
partition the lattice in 4-D over the nodes and exchange the boundary once per application).

Host logic only -- which rank owns what, who the neighbours are, which boundary phase a hop carries, and moving the
face buffers with torch.distributed point-to-point calls (nccl on GPUs, gloo in the CPU tests).  Every arithmetic
step runs in the library's kernels (csrc/halo.cu, csrc/wilson_clover.cu): pack -> [exchange || interior] -> add.
"""
from __future__ import annotations

import numpy as np
import torch

from . import (coarse_bicgstab_hooks, coarse_halo_add, coarse_halo_buffers, coarse_halo_pack, coarse_mult_interior,
               empty_spinor, halo_buffers, mr_domain_solve, mr_workspace, prolong, restrict, wilson_clover_halo_add,
               wilson_clover_halo_pack, wilson_clover_mult_interior, wilson_clover_residual_interior)


class RankGrid:
    """A 4-D grid of ranks, x fastest (rank = c0 + R0 (c1 + R1 (c2 + R2 c3))), periodic like the lattice."""

    def __init__(self, ranks, rank: int = 0):
        self.ranks = tuple(int(r) for r in ranks)
        if len(self.ranks) != 4 or min(self.ranks) < 1:
            raise ValueError(f"rank grid {ranks}")
        self.world = int(np.prod(self.ranks))
        if not 0 <= rank < self.world:
            raise ValueError(f"rank {rank} outside a grid of {self.world}")
        self.rank = int(rank)
        c, r = [], self.rank
        for mu in range(4):
            c.append(r % self.ranks[mu])
            r //= self.ranks[mu]
        self.coords = tuple(c)

    def rank_of(self, coords) -> int:
        r = 0
        for mu in (3, 2, 1, 0):
            r = r * self.ranks[mu] + coords[mu] % self.ranks[mu]
        return r

    def neighbour(self, mu: int, sign: int) -> int:
        c = list(self.coords)
        c[mu] += sign
        return self.rank_of(c)

    @property
    def part_mask(self) -> int:
        """Bit mu set: direction mu is split over more than one rank."""
        return sum(1 << mu for mu in range(4) if self.ranks[mu] > 1)

    def face_phase(self, bc, part_mask=None):
        """face_phase[2 mu + dir] of lqcd_wilson_clover_halo_add: bc[mu] where that hop wraps the global lattice."""
        mask = self.part_mask if part_mask is None else part_mask
        ph = [1] * 8
        for mu in range(4):
            if not (mask >> mu) & 1:
                continue
            if self.coords[mu] == 0:
                ph[2 * mu] = int(bc[mu])                      # backward hop from x_mu = 0
            if self.coords[mu] == self.ranks[mu] - 1:
                ph[2 * mu + 1] = int(bc[mu])                  # forward hop from x_mu = L - 1
        return ph

    def local_dims(self, gdims):
        for mu in range(4):
            if gdims[mu] % self.ranks[mu]:
                raise ValueError(f"global extent {gdims[mu]} not divisible by {self.ranks[mu]} ranks in direction {mu}")
        return tuple(gdims[mu] // self.ranks[mu] for mu in range(4))

    def local_slices(self, gdims):
        """Slices of a canonical field viewed as (L3, L2, L1, L0, ...) that select this rank's sub-lattice."""
        ld = self.local_dims(gdims)
        return tuple(slice(self.coords[mu] * ld[mu], (self.coords[mu] + 1) * ld[mu]) for mu in (3, 2, 1, 0))


def split_field(a, gdims, grid: RankGrid, site_axis: int = 0):
    """This rank's part of a canonical field whose axis `site_axis` runs over the global sites (x fastest)."""
    shp = tuple(a.shape)
    view = a.reshape(shp[:site_axis] + (gdims[3], gdims[2], gdims[1], gdims[0]) + shp[site_axis + 1:])
    idx = (slice(None),) * site_axis + grid.local_slices(gdims)
    loc = view[idx]
    ld = grid.local_dims(gdims)
    loc = loc.reshape(shp[:site_axis] + (int(np.prod(ld)),) + shp[site_axis + 1:])
    return loc.contiguous() if isinstance(loc, torch.Tensor) else np.ascontiguousarray(loc)


def join_field(parts, gdims, ranks, site_axis: int = 0):
    """Inverse of split_field: parts[rank] -> the global canonical field (numpy)."""
    g0 = RankGrid(ranks, 0)
    ld = g0.local_dims(gdims)
    p0 = np.asarray(parts[0])
    shp = p0.shape
    out = np.empty(shp[:site_axis] + (gdims[3], gdims[2], gdims[1], gdims[0]) + shp[site_axis + 1:], dtype=p0.dtype)
    for r, part in enumerate(parts):
        g = RankGrid(ranks, r)
        idx = (slice(None),) * site_axis + g.local_slices(gdims)
        out[idx] = np.asarray(part).reshape(shp[:site_axis] + (ld[3], ld[2], ld[1], ld[0]) + shp[site_axis + 1:])
    return out.reshape(shp[:site_axis] + (int(np.prod(gdims)),) + shp[site_axis + 1:])


def exchange_faces(send, recv, grid: RankGrid, part_mask=None, group=None):
    """recv[2 mu] := send[2 mu + 1] of the -mu neighbour; recv[2 mu + 1] := send[2 mu] of the +mu neighbour.

    Returns the list of the 8 buffers that hold the received faces: `recv[f]`, or -- where the neighbour is this very
    rank -- the send buffer itself (no copy).  Point-to-point operations are posted in one batch, in the same order on
    every rank (per direction: to +mu, to -mu; from -mu, from +mu), so that the two messages between a pair of ranks
    that are each other's neighbour on both sides (two ranks in a direction) match up under nccl's per-peer ordering.
    """
    import torch.distributed as dist
    mask = grid.part_mask if part_mask is None else part_mask
    got = [None] * 8
    ops = []
    for mu in range(4):
        if not (mask >> mu) & 1:
            continue
        plus, minus = grid.neighbour(mu, +1), grid.neighbour(mu, -1)
        if plus == grid.rank and minus == grid.rank:
            got[2 * mu], got[2 * mu + 1] = send[2 * mu + 1], send[2 * mu]
            continue
        ops.append(dist.P2POp(dist.isend, send[2 * mu + 1], plus, group=group, tag=2 * mu))
        ops.append(dist.P2POp(dist.isend, send[2 * mu], minus, group=group, tag=2 * mu + 1))
        ops.append(dist.P2POp(dist.irecv, recv[2 * mu], minus, group=group, tag=2 * mu))
        ops.append(dist.P2POp(dist.irecv, recv[2 * mu + 1], plus, group=group, tag=2 * mu + 1))
        got[2 * mu], got[2 * mu + 1] = recv[2 * mu], recv[2 * mu + 1]
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    return got


def route_faces(sends, ranks, part_mask):
    """Single-process stand-in for exchange_faces: sends[rank][8] -> recvs[rank][8] by reference (no copies).
    Used where several virtual ranks live on one GPU one after the other (tests, the bench's overhead probe)."""
    recvs = []
    for r in range(len(sends)):
        g = RankGrid(ranks, r)
        got = [None] * 8
        for mu in range(4):
            if (part_mask >> mu) & 1:
                got[2 * mu] = sends[g.neighbour(mu, -1)][2 * mu + 1]
                got[2 * mu + 1] = sends[g.neighbour(mu, +1)][2 * mu]
        recvs.append(got)
    return recvs


class PeerFaces:
    """The receive faces of this rank in ONE symmetric-memory allocation (torch.distributed._symmetric_memory), twice
    (double-buffered), every rank's copy mapped into every other rank's address space over NVLink.

    With it the exchange is no separate step: the pack kernel is handed, as its `send[8]`, the NEIGHBOURS' receive
    buffers, so its stores are the transfer (compute and communication in one kernel, face site by face site), and
    what remains is one device-side barrier (`arrive`, stream-ordered) before the add kernel may read.  Double
    buffering makes that one barrier per application enough: a rank can write application n + 2 only after every
    rank has passed barrier n + 1, which each rank enqueues after its add kernel of application n.
    `face_reals[f]`: reals of face f (0 where the direction is not partitioned)."""

    def __init__(self, face_reals, dtype, device, grid: RankGrid, group=None):
        import torch.distributed as dist
        import torch.distributed._symmetric_memory as symm
        off, total = [], 0
        for n in face_reals:
            off.append(total)
            total += (int(n) + 3) // 4 * 4                       # keep every face 16-byte aligned
        self.total = total
        self.buf = symm.empty(2 * total, dtype=dtype, device=device)
        self.hdl = symm.rendezvous(self.buf, dist.group.WORLD if group is None else group)
        if self.hdl.rank != grid.rank or self.hdl.world_size != grid.world:
            raise ValueError("the rank grid must enumerate the ranks of the group")
        self.send, self.recv, self.parity = [[None] * 8, [None] * 8], [[None] * 8, [None] * 8], 0
        for par in range(2):
            base = par * total
            for mu in range(4):
                lo, hi = 2 * mu, 2 * mu + 1
                if not face_reals[lo]:
                    continue
                n = (int(face_reals[lo]),)
                plus, minus = grid.neighbour(mu, +1), grid.neighbour(mu, -1)
                self.recv[par][lo] = self.hdl.get_buffer(grid.rank, n, dtype, base + off[lo])
                self.recv[par][hi] = self.hdl.get_buffer(grid.rank, n, dtype, base + off[hi])
                # my forward face feeds the +mu neighbour's recv[2 mu]; my backward face the -mu neighbour's recv[2 mu + 1]
                self.send[par][hi] = self.hdl.get_buffer(plus, n, dtype, base + off[lo])
                self.send[par][lo] = self.hdl.get_buffer(minus, n, dtype, base + off[hi])

    def next(self):
        par, self.parity = self.parity, self.parity ^ 1
        return self.send[par], self.recv[par]

    def arrive(self):
        """Every rank's stores issued before this point (on the stream it is called under) are visible after it."""
        self.hdl.barrier(channel=0)


class ShardedWilsonClover:
    """D (or D^dag) on this rank's sub-lattice of a lattice split over `grid`.

    U, clover: this rank's native fields (lattice `dims` = the LOCAL extents).  part_mask defaults to the directions
    the grid really splits; a direction may also be marked partitioned with a single rank in it (the rank is then
    its own neighbour) -- the result is the same operator, which is how one GPU exercises the whole exchange path.
    """

    def __init__(self, U, clover, kappa, dims, bc, grid: RankGrid, links12=False, part_mask=None, group=None,
                 transport="p2p", exchange=None):
        """transport: "p2p" = pack into local buffers, torch.distributed send/recv; "peer" = the pack kernel stores
        straight into the neighbours' receive buffers over NVLink peer memory (PeerFaces)."""
        self.U, self.clover, self.kappa = U, clover, float(kappa)
        self.dims, self.bc, self.grid, self.links12, self.group = tuple(dims), tuple(bc), grid, links12, group
        self.exchange = exchange_faces if exchange is None else exchange   # (send, recv, grid, mask, group) -> got
        self.mask = grid.part_mask if part_mask is None else int(part_mask)
        if grid.part_mask & ~self.mask:
            raise ValueError("part_mask must include every direction the rank grid splits")
        self.phase = grid.face_phase(bc, self.mask)
        self.send = halo_buffers(dims, self.mask, dtype=U.dtype, device=U.device)
        remote = [mu for mu in range(4) if (self.mask >> mu) & 1 and grid.neighbour(mu, 1) != grid.rank]
        rmask = sum(1 << mu for mu in remote)
        self.recv = halo_buffers(dims, rmask, dtype=U.dtype, device=U.device)
        self.comm = torch.cuda.Stream(device=U.device)
        self.peer = None
        if transport == "peer":
            from . import halo_face_reals
            self.peer = PeerFaces([halo_face_reals(dims, f >> 1) if (self.mask >> (f >> 1)) & 1 else 0
                                   for f in range(8)], U.dtype, U.device, grid, group)
        elif transport != "p2p":
            raise ValueError(f"transport {transport!r}")

    def _run(self, out, inp, dagger, rhs, domain=None, parity=0):
        cur = torch.cuda.current_stream(self.U.device)
        send, got = (self.send, None) if self.peer is None else self.peer.next()
        wilson_clover_halo_pack(send, inp, self.U, self.dims, self.mask, dagger, self.links12, stream=cur)
        packed = cur.record_event()
        with torch.cuda.stream(self.comm):           # the exchange overlaps the interior pass
            self.comm.wait_event(packed)
            if self.peer is None:
                got = self.exchange(self.send, self.recv, self.grid, self.mask, self.group)
            else:
                self.peer.arrive()
            arrived = self.comm.record_event()
        if rhs is None:
            wilson_clover_mult_interior(out, inp, self.U, self.clover, self.kappa, self.dims, self.bc, self.mask,
                                        dagger, self.links12, stream=cur)
        else:
            wilson_clover_residual_interior(out, rhs, inp, self.U, self.clover, self.kappa, self.dims, self.bc,
                                            self.mask, self.links12, domain, parity, stream=cur)
        cur.wait_event(arrived)
        # the residual carries -D: the faces enter with the opposite sign
        wilson_clover_halo_add(out, got, self.U, self.kappa if rhs is None else -self.kappa, self.dims, self.phase,
                               self.mask, dagger, self.links12, stream=cur)
        return out

    def apply(self, out, inp, dagger=False):
        """out = D inp (or D^dag inp)."""
        return self._run(out, inp, dagger, None)

    def residual(self, r, b, x, domain=None, parity=0):
        """r = b - D x; r must not alias b or x.  parity 1 / 2 with a domain: only on the
        even / odd domains (LOCAL colouring) -- the rest of r is then not meaningful."""
        return self._run(r, x, False, b, domain, parity)


class ShardedSAP:
    """The SAP smoother with fixed iterations (lqcd_sap, Q17) on a lattice split over
    ranks: the domain solves M_SAP^(e/o) are local -- "D_SAP needs no communication", PAPER.md:125 -- and only the
    residual r = b - D x between the half sweeps exchanges halos.  Same sequence of kernels as lqcd_sap on one GPU.

    The even/odd colouring of the domains is that of the GLOBAL lattice: a rank whose corner sits at an odd domain
    coordinate sum swaps the two groups.  Every partitioned direction must hold at least two domains per rank (a
    single domain would be joined to itself around the local lattice)."""

    def __init__(self, op: ShardedWilsonClover, domain, n_sap=4, n_mr=6):
        self.op, self.domain, self.n_sap, self.n_mr = op, tuple(int(d) for d in domain), int(n_sap), int(n_mr)
        self.flip = domain_parity_flip(op.grid, op.dims, self.domain, op.mask)
        self.ws = mr_workspace(op.dims, self.domain, dtype=op.U.dtype, device=op.U.device)

    def apply(self, x, r, b, initial_guess=False, final_residual=True):
        """x = SAP_n(b) (or x + SAP_n(b - D x) with initial_guess); r: scratch, receives b - D x."""
        op = self.op
        # between two half sweeps only the group solved next reads the residual (as in lqcd_sap)
        group = lambda g: 1 + (g ^ self.flip)
        if initial_guess:
            op.residual(r, b, x, self.domain, group(0) if self.n_sap > 0 else 0)
            res = r
        else:
            x.zero_()
            res = b
            if self.n_sap == 0 and final_residual:
                r.copy_(b)
        for i in range(self.n_sap):
            for g in (0, 1):
                mr_domain_solve(x, res, op.U, op.clover, op.kappa, op.dims, op.bc, self.domain,
                                parity=group(g), niter=self.n_mr, accumulate=True, ws=self.ws)
                last = i == self.n_sap - 1 and g == 1
                if last and not final_residual:
                    break
                op.residual(r, b, x, self.domain, 0 if last else group(g ^ 1))
                res = r
        return x


def domain_parity_flip(grid: RankGrid, dims, domain, part_mask=None) -> int:
    """1 if this rank's local even domains are the global odd ones (its corner has an odd domain-coordinate sum)."""
    mask = grid.part_mask if part_mask is None else part_mask
    off = 0
    for mu in range(4):
        if dims[mu] % domain[mu]:
            raise ValueError(f"domain extent {domain[mu]} does not divide the local extent {dims[mu]}")
        n = dims[mu] // domain[mu]
        if (mask >> mu) & 1 and n < 2:
            raise ValueError(f"direction {mu} is partitioned but holds only {n} domain per rank")
        off += grid.coords[mu] * n
    return off & 1


class ShardedCoarse:
    """D_c (or its dagger) on this rank's part of a coarse lattice split over `grid`; A: the blocks of the local sites.
    cdims = the LOCAL coarse extents.  No boundary phases: bc lives inside A."""

    def __init__(self, A, cdims, nvec, grid: RankGrid, part_mask=None, group=None, transport="p2p", exchange=None):
        self.A, self.cdims, self.nvec, self.grid, self.group = A, tuple(cdims), int(nvec), grid, group
        self.exchange = exchange_faces if exchange is None else exchange
        self.mask = grid.part_mask if part_mask is None else int(part_mask)
        if grid.part_mask & ~self.mask:
            raise ValueError("part_mask must include every direction the rank grid splits")
        rdt = torch.float32 if A.dtype in (torch.complex64, torch.float32) else torch.float64
        self.send = coarse_halo_buffers(cdims, nvec, self.mask, dtype=rdt, device=A.device)
        rmask = sum(1 << mu for mu in range(4) if (self.mask >> mu) & 1 and grid.neighbour(mu, 1) != grid.rank)
        self.recv = coarse_halo_buffers(cdims, nvec, rmask, dtype=rdt, device=A.device)
        self.comm = torch.cuda.Stream(device=A.device)
        self.peer = None
        if transport == "peer":
            from . import coarse_halo_face_reals
            self.peer = PeerFaces([coarse_halo_face_reals(cdims, nvec, f >> 1) if (self.mask >> (f >> 1)) & 1 else 0
                                   for f in range(8)], rdt, A.device, grid, group)
        elif transport != "p2p":
            raise ValueError(f"transport {transport!r}")

    def apply(self, out, inp, dagger=False):
        cur = torch.cuda.current_stream(self.A.device)
        send, got = (self.send, None) if self.peer is None else self.peer.next()
        coarse_halo_pack(send, inp, self.cdims, self.nvec, self.mask, stream=cur)
        packed = cur.record_event()
        with torch.cuda.stream(self.comm):
            self.comm.wait_event(packed)
            if self.peer is None:
                got = self.exchange(self.send, self.recv, self.grid, self.mask, self.group)
            else:
                self.peer.arrive()
            arrived = self.comm.record_event()
        coarse_mult_interior(out, inp, self.A, self.cdims, self.nvec, self.mask, dagger, stream=cur)
        cur.wait_event(arrived)
        coarse_halo_add(out, got, self.A, self.cdims, self.nvec, self.mask, dagger, stream=cur)
        return out


def allreduce_sum(group=None):
    """The cross-rank sum for ShardedVcycle / coarse_bicgstab_hooks: an in-place torch.distributed all-reduce (nccl:
    ordered on the current stream), or None when there is one rank."""
    import torch.distributed as dist
    if not dist.is_available() or not dist.is_initialized() or dist.get_world_size(group) == 1:
        return None
    return lambda t: dist.all_reduce(t, group=group)


class ShardedVcycle:
    """x = M b, one V-cycle of the multigrid preconditioner (lqcd_mg_vcycle, Q19) on a
    lattice split over ranks: restrict (block-local) -> fixed-iteration BiCGStab on the sharded D_c, its dot products
    summed over the ranks (`reduce`) -> prolong (block-local) -> SAP started from that x (ShardedSAP).
    nullvecs: the native null vectors of this rank's aggregates; the smoother's domains are the aggregates."""

    def __init__(self, fine: ShardedWilsonClover, coarse: ShardedCoarse, nullvecs, block, nvec, n_coarse=8, n_sap=4,
                 n_mr=6, reduce=None):
        self.fine, self.coarse, self.v = fine, coarse, nullvecs
        self.block, self.nvec, self.n_coarse = tuple(int(v) for v in block), int(nvec), int(n_coarse)
        # more than one rank and no sum given: the process group's all-reduce
        self.reduce = allreduce_sum(fine.group) if reduce is None and fine.grid.world > 1 else reduce
        self.sap = ShardedSAP(fine, self.block, n_sap, n_mr)
        cdt = torch.complex64 if fine.U.dtype == torch.float32 else torch.complex128
        vc = int(np.prod(coarse.cdims))
        self.bc_ = torch.empty((vc, 2, self.nvec), dtype=cdt, device=fine.U.device)
        self.xc_ = torch.empty_like(self.bc_)
        self.r_ = empty_spinor(fine.dims, dtype=fine.U.dtype, device=fine.U.device)

    def apply(self, x, b):
        f, c = self.fine, self.coarse
        restrict(self.bc_, b, self.v, f.dims, self.block, self.nvec)                                     # (1a) Eq. 5
        coarse_bicgstab_hooks(self.xc_, self.bc_, c.cdims, self.nvec, self.n_coarse,                     # (1b)
                              apply=lambda o, i: c.apply(o, i), reduce=self.reduce)
        prolong(x, self.xc_, self.v, f.dims, self.block, self.nvec)                                      # (1c) Eq. 6
        if self.sap.n_sap > 0:                                                                           # (2)
            self.sap.apply(x, self.r_, b, initial_guess=True, final_residual=False)
        return x

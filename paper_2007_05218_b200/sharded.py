"""Box sharding of one MultiFab over several GPUs: every rank owns a contiguous
block of the box grid, i.e. a sub-domain with its own handle of the C ABI; faces between ranks carry the
boundary type HYDRO_BC_EXTERNAL, whose ghost zones are filled by a halo exchange instead of by
hydro_fill_ghosts.  Per RK stage: local ghost fill, then one exchange per dimension (x, then y, then z), each
sending the `ng` valid layers next to a face over the FULL padded extent of the other two dimensions, so that
edges and corners arrive through the earlier dimensions' ghosts (6 messages per rank and stage instead of 26).
Per step: one allreduce-min of dt (8 bytes).  Totals: one allreduce-sum of NFLUX doubles.

Plumbing only: packing, unpacking and every step of the path run in the library's kernels
(hydro_pack_halo / hydro_unpack_halo, include/hydro.h); the transfers are torch.distributed point-to-point
operations (NCCL over NVLink between GPUs; gloo with host tensors in the CPU tests) or, for several shards held
by ONE process on one device (the single-GPU validation of this module), plain tensor copies.
"""
from __future__ import annotations

import copy

BC_EXTERNAL = 3


def proc_coords(rank: int, pgrid):
    """rank -> (px, py, pz), x fastest."""
    px = rank % pgrid[0]
    py = (rank // pgrid[0]) % pgrid[1]
    pz = rank // (pgrid[0] * pgrid[1])
    return px, py, pz


def proc_rank(coords, pgrid):
    return (coords[2] * pgrid[1] + coords[1]) * pgrid[0] + coords[0]


def local_params(params: dict, pgrid, rank: int):
    """The hydro_params of rank's sub-domain and its neighbours: ({params}, {(dim, side): neighbour rank}).
    A dimension is cut into pgrid[d] equal blocks of whole boxes.  A face shared with another rank (inside the
    domain, or across a periodic boundary of a dimension that is cut) becomes HYDRO_BC_EXTERNAL."""
    p = copy.deepcopy(params)
    c = proc_coords(rank, pgrid)
    nbrs = {}
    for d in range(3):
        P = pgrid[d]
        nboxes = params["ndom"][d] // params["nbox"][d]
        if params["ndom"][d] % params["nbox"][d] or nboxes % P:
            raise ValueError(f"dimension {d}: {nboxes} boxes cannot be cut into {P} equal blocks")
        n = params["ndom"][d] // P
        dx = params.get("dx", (0.0, 0.0, 0.0))[d] or (params["prob_hi"][d] - params["prob_lo"][d]) / params["ndom"][d]
        p["ndom"][d] = n
        p["prob_lo"][d] = params["prob_lo"][d] + c[d] * n * dx
        p["prob_hi"][d] = params["prob_lo"][d] + (c[d] + 1) * n * dx
        # the zone width of the UNSHARDED domain, bit for bit: (prob_hi - prob_lo)/n of the piece is off by an ulp for
        # a third of the non-dyadic spacings, and the shards would then differ from the unsharded run and each other
        p["dx"] = list(p.get("dx", (0.0, 0.0, 0.0)))
        p["dx"][d] = p["dx"][d] or dx
        if P == 1:
            continue
        periodic = params["bc_lo"][d] == 0
        for side, step in ((0, -1), (1, +1)):
            q = c[d] + step
            if 0 <= q < P or periodic:
                cc = list(c)
                cc[d] = q % P
                nbrs[(d, side)] = proc_rank(cc, pgrid)
                p["bc_lo" if side == 0 else "bc_hi"][d] = BC_EXTERNAL
    return p, nbrs


def exchange_plan(nbrs, dim):
    """[(side to send from, destination rank, side the neighbour unpacks into)] of one dimension: the layers
    next to MY low face become the neighbour's HIGH ghosts and vice versa."""
    return [(side, nbrs[(dim, side)], 1 - side) for side in (0, 1) if (dim, side) in nbrs]


def exchange_dim(dim, nbrs, pack, unpack, sendrecv):
    """One dimension of the halo exchange of one rank.  pack(dim, side) -> buffer of my valid layers next to
    `side`; unpack(dim, side, buffer) fills my ghost layers beyond `side`; sendrecv([(send buffer, dst rank, tag)],
    [(src rank, tag)]) -> received buffers in the order of the second list."""
    plan = exchange_plan(nbrs, dim)
    # Sends go out low side first.  A dimension cut in two with periodic wrap has BOTH messages of a rank going to
    # the same peer; NCCL ignores tags and pairs the sends and receives of two ranks in posting order, so the
    # receives are posted in the order of the peer's sends: its low-side message fills MY high ghosts, hence high
    # side first.  The tag (the side of the RECEIVER the message is for) says the same to backends that honour tags.
    sends = [(pack(dim, side), dst, 2 * dim + (1 - side)) for side, dst, _ in plan]
    sides = [side for side, _, _ in reversed(plan)]
    recvs = [(nbrs[(dim, side)], 2 * dim + side) for side in sides]
    for side, buf in zip(sides, sendrecv(sends, recvs)):
        unpack(dim, side, buf)


def dist_sendrecv(like, stage_on_host=False):
    """sendrecv over torch.distributed point-to-point operations (one batch per call).  stage_on_host: copy the
    buffers through host memory (for the gloo backend, which moves host tensors; NCCL sends device buffers)."""
    import torch
    import torch.distributed as dist

    def f(sends, recvs):
        dev = [like(src, tag) for src, tag in recvs]
        outs = [torch.empty_like(d, device="cpu" if stage_on_host else d.device) for d in dev]
        ops = [dist.P2POp(dist.isend, buf.cpu() if stage_on_host else buf, dst, tag=tag) for buf, dst, tag in sends]
        ops += [dist.P2POp(dist.irecv, out, src, tag=tag) for out, (src, tag) in zip(outs, recvs)]
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()
        return [o.to(d.device) for o, d in zip(outs, dev)] if stage_on_host else outs
    return f


class Shard:
    """One rank's sub-domain: a Hydro handle plus the pack / unpack calls of its halos."""

    def __init__(self, params: dict, pgrid, rank: int, device="cuda:0"):
        from .binding import Hydro, hydro_halo_bytes, make_params
        self.rank, self.pgrid = rank, tuple(pgrid)
        self.params, self.nbrs = local_params(params, pgrid, rank)
        self.h = Hydro(self.params, device=device)
        p = make_params(self.params)
        import torch
        self.bufs = {(d, s): torch.empty(hydro_halo_bytes(p, d) // 8, dtype=torch.float64, device=device)
                     for (d, s) in self.nbrs}

    def pack(self, which):
        def f(dim, side):
            self.h.hydro_pack_halo(which, dim, side, self.bufs[(dim, side)])
            return self.bufs[(dim, side)]
        return f

    def unpack(self, which):
        return lambda dim, side, buf: self.h.hydro_unpack_halo(which, dim, side, buf)


class ShardedHydro:
    """All-ranks driver of one process per GPU (torch.distributed must be initialised; backend nccl)."""

    def __init__(self, params: dict, pgrid, device):
        import torch.distributed as dist
        self.dist = dist
        self.on_host = dist.get_backend() == "gloo"            # gloo: buffers and scalars go through host memory
        self.shard = Shard(params, pgrid, dist.get_rank(), device=device)
        self.sendrecv = dist_sendrecv(lambda src, tag: self.shard.bufs[(tag // 2, tag % 2)], stage_on_host=self.on_host)

    def fill(self, which):
        s = self.shard
        s.h.hydro_fill_ghosts(which)
        for dim in range(3):
            s.h.torch.cuda.current_stream(s.h.device).synchronize()
            exchange_dim(dim, s.nbrs, s.pack(which), s.unpack(which), self.sendrecv)

    def step(self):
        import torch
        s = self.shard
        dt = torch.tensor([s.h.hydro_estimate_dt()], dtype=torch.float64, device="cpu" if self.on_host else s.h.device)
        self.dist.all_reduce(dt, op=self.dist.ReduceOp.MIN)          # the one collective of a step: 8 bytes
        dt = float(dt.item())
        self.fill(0)
        s.h.hydro_advance_stage(0, dt)
        self.fill(1)
        s.h.hydro_advance_stage(1, dt)
        return dt

    def totals(self):
        import torch
        t = torch.tensor(self.shard.h.hydro_conserved_totals(0), dtype=torch.float64,
                         device="cpu" if self.on_host else self.shard.h.device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        return t.tolist()


class LocalShards:
    """Every shard of the decomposition in ONE process on one device: the exchange is a tensor copy.  This is the
    validation harness of the sharded path on a single GPU (results must equal the unsharded run bit for bit);
    it runs the shards one after the other, never concurrently."""

    def __init__(self, params: dict, pgrid, device="cuda:0"):
        self.pgrid = tuple(pgrid)
        self.shards = [Shard(params, pgrid, r, device=device) for r in range(pgrid[0] * pgrid[1] * pgrid[2])]

    def fill(self, which):
        for s in self.shards:
            s.h.hydro_fill_ghosts(which)
        for dim in range(3):
            packed = {}
            for s in self.shards:                                     # everybody packs, then everybody unpacks
                for side, dst, dside in exchange_plan(s.nbrs, dim):
                    packed[(dst, dside)] = s.pack(which)(dim, side).clone()
            for s in self.shards:
                for side in (0, 1):
                    if (dim, side) in s.nbrs:
                        s.unpack(which)(dim, side, packed[(s.rank, side)])

    def step(self):
        dt = min(s.h.hydro_estimate_dt() for s in self.shards)
        self.fill(0)
        for s in self.shards:
            s.h.hydro_advance_stage(0, dt)
        self.fill(1)
        for s in self.shards:
            s.h.hydro_advance_stage(1, dt)
        return dt

    def totals(self):
        import numpy as np
        return np.sum([s.h.hydro_conserved_totals(0) for s in self.shards], axis=0).tolist()

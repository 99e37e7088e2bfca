"""Host logic of the box sharding (paper_2007_05218_b200/sharded.py) on CPU: the
decomposition into sub-domains, the neighbour table, and the dimension-by-dimension halo exchange over two and
four gloo ranks.  The device kernels cannot run here, so pack / unpack are numpy slices of the same layers
(test code); the local ghost fill is the oracle's with OUTFLOW at the faces shared with another rank (every such
ghost layer is then overwritten by the exchange).  After the exchange every zone of every rank's padded state,
ghosts, edges and corners included, must equal the oracle's ghost fill of the UNSHARDED domain."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2007_05218_b200 import sharded as S  # noqa: E402
from paper_2007_05218_b200 import workloads as W  # noqa: E402


def test_local_params_and_neighbours():
    wl = W.config(5, ndom=(64, 64, 64), nbox=(16, 16, 16))
    p, nb = S.local_params(wl.params, (2, 1, 2), 3)                      # rank 3 = (px 1, py 0, pz 1)
    assert p["ndom"] == [32, 64, 32] and p["nbox"] == [16, 16, 16]
    assert p["prob_lo"] == [0.5, 0.0, 0.5] and p["prob_hi"] == [1.0, 1.0, 1.0]
    assert p["bc_lo"] == [3, 0, 3] and p["bc_hi"] == [3, 0, 3]            # periodic y stays local, x and z are cut
    assert nb == {(0, 0): 2, (0, 1): 2, (2, 0): 1, (2, 1): 1}             # periodic wrap: both sides the same rank
    wl4 = W.config(4, ndom=(32, 32, 64), nbox=(16, 16, 16))               # reflecting z walls
    p, nb = S.local_params(wl4.params, (1, 1, 4), 0)
    assert p["bc_lo"][2] == 2 and p["bc_hi"][2] == 3 and nb == {(2, 1): 1}
    p, nb = S.local_params(wl4.params, (1, 1, 4), 3)
    assert p["bc_lo"][2] == 3 and p["bc_hi"][2] == 2 and nb == {(2, 0): 2}
    with pytest.raises(ValueError):
        S.local_params(wl.params, (3, 1, 1), 0)
    assert [S.proc_rank(S.proc_coords(r, (2, 3, 2)), (2, 3, 2)) for r in range(12)] == list(range(12))


@pytest.mark.parametrize("pgrid,periodic", [((2, 1, 1), True), ((2, 2, 2), True), ((3, 1, 2), True), ((2, 1, 4), False)])
def test_exchange_matches_by_posting_order_alone(pgrid, periodic):
    """ProcessGroupNCCL ignores P2P tags: between two ranks the n-th send meets the n-th receive.  Model exactly
    that (one FIFO per ordered pair of ranks, tags dropped) and run exchange_dim for every rank of the grid: the
    ghost layers beyond my `side` must come from my neighbour's OPPOSITE side, also where a periodic dimension is cut
    in two and both of a rank's messages go to the same peer."""
    wl = W.config(5, ndom=(96, 32, 64), nbox=(16, 16, 16))
    params = dict(wl.params)
    if not periodic:
        params["bc_lo"], params["bc_hi"] = [1, 1, 1], [1, 1, 1]
    world = pgrid[0] * pgrid[1] * pgrid[2]
    nbrs = [S.local_params(params, pgrid, r)[1] for r in range(world)]
    for dim in range(3):
        fifo = {}

        def post(rank):          # pass 1: every rank posts its sends (payload = who packed it, from which side)
            def sendrecv(sends, recvs):
                for buf, dst, _tag in sends:
                    fifo.setdefault((rank, dst), []).append(buf)
                return [None] * len(recvs)
            return sendrecv

        def match(rank):         # pass 2: the same posting order again, receives served from the FIFOs
            def sendrecv(sends, recvs):
                return [fifo[(src, rank)].pop(0) for src, _tag in recvs]
            return sendrecv

        for r in range(world):
            S.exchange_dim(dim, nbrs[r], lambda d, s, r=r: (r, s), lambda d, s, buf: None, post(r))
        got = {}
        for r in range(world):
            S.exchange_dim(dim, nbrs[r], lambda d, s, r=r: (r, s),
                           lambda d, s, buf, r=r: got.__setitem__((r, s), buf), match(r))
        assert all(not q for q in fifo.values())
        want = {(r, s): (nbrs[r][(dim, s)], 1 - s) for r in range(world) for s in (0, 1) if (dim, s) in nbrs[r]}
        assert got == want


def test_shards_carry_the_global_zone_width_exactly():
    """(prob_hi - prob_lo)/ndom of a piece of a non-dyadic domain is off by an ulp in many cases (48 zones over
    [0.1, 1.3] cut in two is one), and a shard with another dx no longer gives the bits of the unsharded run:
    local_params hands every shard the unsharded zone width in hydro_params.dx, which the library then uses instead
    of the quotient.  The library rejects a negative or non-finite dx."""
    from paper_2007_05218_b200 import binding as B
    from paper_2007_05218_b200 import build as build_mod
    wl = W.config(5, ndom=(48, 24, 24), nbox=(12, 12, 12), nspec=2)
    wl.params["prob_lo"], wl.params["prob_hi"] = [0.1, 0.1, 0.1], [1.3, 0.7, 0.7]
    dx = [(wl.params["prob_hi"][d] - wl.params["prob_lo"][d]) / wl.params["ndom"][d] for d in range(3)]
    off = 0
    for r in range(4):
        p, _ = S.local_params(wl.params, (2, 2, 1), r)
        assert p["dx"] == dx                                                          # all three, cut or not
        off += (p["prob_hi"][0] - p["prob_lo"][0]) / p["ndom"][0] != dx[0]
        assert B.make_params(p).dx[0] == dx[0]
    assert off > 0                     # the case is one where the piece's own quotient would have been wrong
    build_mod.build()
    assert B.hydro_state_bytes(B.make_params(p)) > 0
    for bad in (-1.0, float("inf"), float("nan")):
        q = dict(p, dx=[bad, 0.0, 0.0])
        assert B.hydro_state_bytes(B.make_params(q)) == 0


# ---- numpy stand-ins of hydro_pack_halo / hydro_unpack_halo on a (boxes, nvar, nt2, nt1, nt0) state --------------
def np_pack(U, wl, dim, side):
    """the ng valid layers next to `side` of dimension dim of the boxes on that face, full padded extent elsewhere"""
    ng, nb, NB = wl.ng, wl.nb, wl.NB
    out = []
    for b in range(wl.nboxes):
        c = (b % NB[0], (b // NB[0]) % NB[1], b // (NB[0] * NB[1]))
        if c[dim] != (0 if side == 0 else NB[dim] - 1):
            continue
        lo = ng if side == 0 else nb[dim]
        sl = [slice(None)] * 4
        sl[3 - dim] = slice(lo, lo + ng)
        out.append(U[b][tuple(sl)].copy())
    return np.stack(out)


def np_unpack(U, wl, dim, side, buf):
    ng, nb, NB = wl.ng, wl.nb, wl.NB
    i = 0
    for b in range(wl.nboxes):
        c = (b % NB[0], (b // NB[0]) % NB[1], b // (NB[0] * NB[1]))
        if c[dim] != (0 if side == 0 else NB[dim] - 1):
            continue
        lo = 0 if side == 0 else nb[dim] + ng
        sl = [slice(None)] * 4
        sl[3 - dim] = slice(lo, lo + ng)
        U[b][tuple(sl)] = buf[i]
        i += 1


def _rank_main(rank, world, port, pgrid, bcs, q):
    import torch
    import torch.distributed as dist
    from oracle import oracle_binding as O
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = W.uniform((32, 16, 24), (8, 8, 6), 2, (1, 0, 0, 0, 1), bc=bcs)
    # index-encoded global state: every valid zone of every component carries its own global identity
    rng = np.random.default_rng(7)
    Gglob = rng.standard_normal((wl.nvar, 24, 16, 32))
    Uglob = W.scatter_valid(wl, Gglob, ghost_value=np.nan)
    O.fill_ghosts(O.make_params(wl.params), Uglob)
    # my sub-domain
    lp, nbrs = S.local_params(wl.params, pgrid, rank)
    c = S.proc_coords(rank, pgrid)
    n = lp["ndom"]
    Gloc = Gglob[:, c[2] * n[2]:(c[2] + 1) * n[2], c[1] * n[1]:(c[1] + 1) * n[1], c[0] * n[0]:(c[0] + 1) * n[0]]
    wloc = W.Workload("shard", "uniform", lp, 1, extra=wl.extra)
    U = W.scatter_valid(wloc, Gloc, ghost_value=np.nan)
    op = dict(lp)
    op["bc_lo"] = [1 if b == S.BC_EXTERNAL else b for b in lp["bc_lo"]]   # local fill: outflow where a neighbour rank is
    op["bc_hi"] = [1 if b == S.BC_EXTERNAL else b for b in lp["bc_hi"]]
    O.fill_ghosts(O.make_params(op), U)
    Ub = U.reshape(wloc.state_shape)

    def sendrecv(sends, recvs):
        shapes = {}
        for dim in range(3):
            for side in (0, 1):
                shapes[2 * dim + side] = np_pack(Ub, wloc, dim, side).shape
        outs = [torch.empty(shapes[tag], dtype=torch.float64) for _, tag in recvs]
        ops = [dist.P2POp(dist.isend, torch.from_numpy(np.ascontiguousarray(buf)), dst, tag=tag) for buf, dst, tag in sends]
        ops += [dist.P2POp(dist.irecv, out, src, tag=tag) for out, (src, tag) in zip(outs, recvs)]
        for req in (dist.batch_isend_irecv(ops) if ops else []):
            req.wait()
        return [o.numpy() for o in outs]

    for dim in range(3):
        S.exchange_dim(dim, nbrs, lambda d, s: np_pack(Ub, wloc, d, s), lambda d, s, buf: np_unpack(Ub, wloc, d, s, buf),
                       sendrecv)
    # compare with the unsharded fill, box by box
    ok = True
    Ug = Uglob.reshape(wl.state_shape)
    for b in range(wloc.nboxes):
        lb = (b % wloc.NB[0], (b // wloc.NB[0]) % wloc.NB[1], b // (wloc.NB[0] * wloc.NB[1]))
        gb = [c[d] * wloc.NB[d] + lb[d] for d in range(3)]
        ok = ok and np.array_equal(Ub[b], Ug[(gb[2] * wl.NB[1] + gb[1]) * wl.NB[0] + gb[0]])
    q.put((rank, bool(ok)))
    dist.destroy_process_group()


@pytest.mark.parametrize("pgrid,bcs", [((2, 1, 1), (0, 0, 0)), ((1, 1, 2), (1, 0, 2)), ((2, 1, 2), (0, 2, 0)),
                                       ((1, 2, 2), (1, 1, 1))])
def test_halo_exchange_over_gloo_ranks(pgrid, bcs):
    import torch.multiprocessing as mp
    world = pgrid[0] * pgrid[1] * pgrid[2]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31000 + (os.getpid() + hash((pgrid, bcs))) % 2000
    procs = [ctx.Process(target=_rank_main, args=(r, world, port, pgrid, bcs, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(r, True) for r in range(world)]

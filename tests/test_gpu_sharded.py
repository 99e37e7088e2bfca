"""Box sharding with halo exchange (paper_2007_05218_b200/sharded.py) on ONE GPU: every
shard of a decomposition is a handle of its own on the same device, driven one after the other, the halos go
through hydro_pack_halo / hydro_unpack_halo and a device copy.  The sharded run must reproduce the unsharded
run BIT FOR BIT on every valid zone (the scheme is decomposition invariant, pin P8), with the same dt; totals
agree to rounding (a different reduction tree).  The ghost zones after a sharded fill equal the unsharded fill's."""
import numpy as np
import pytest

from paper_2007_05218_b200 import workloads as W

pytestmark = pytest.mark.gpu

def nondyadic():
    """48 zones over [0.1, 1.3]: the zone width of half the domain, derived from the half's own extent, differs from
    the unsharded zone width by an ulp; the shards must use the unsharded one (hydro_params.dx)."""
    wl = W.config(5, ndom=(48, 24, 24), nbox=(12, 12, 12), nspec=2)
    wl.params["prob_lo"], wl.params["prob_hi"] = [0.1, 0.1, 0.1], [1.3, 0.7, 0.7]
    return wl


CASES = [
    ("cfg5 periodic on a non-dyadic domain, cut in x and y", nondyadic, (2, 2, 1)),
    ("cfg5 periodic, cut in x", lambda: W.config(5, ndom=(64, 32, 32), nbox=(16, 16, 16), nspec=3), (2, 1, 1)),
    ("cfg5 periodic, cut in z (4 slabs)", lambda: W.config(5, ndom=(32, 32, 64), nbox=(16, 16, 16), nspec=2), (1, 1, 4)),
    ("cfg5 periodic, 2x2x2 blocks", lambda: W.config(5, ndom=(64, 64, 64), nbox=(16, 16, 16), nspec=13), (2, 2, 2)),
    ("cfg4 gravity + reflecting z walls, cut in y and z", lambda: W.config(4, ndom=(32, 32, 64), nbox=(16, 16, 16), nspec=2), (1, 2, 2)),
    ("cfg2 Sedov with outflow walls, cut in x and y", lambda: W.config(2, ndom=(48, 48, 48), nbox=(24, 24, 48)), (2, 2, 1)),
]


def shard_blocks(wl, pgrid):
    """(rank, slices of the global valid array) of every shard"""
    from paper_2007_05218_b200 import sharded as S
    n = [wl.params["ndom"][d] // pgrid[d] for d in range(3)]
    for r in range(pgrid[0] * pgrid[1] * pgrid[2]):
        c = S.proc_coords(r, pgrid)
        yield r, (slice(None), slice(c[2] * n[2], (c[2] + 1) * n[2]), slice(c[1] * n[1], (c[1] + 1) * n[1]),
                  slice(c[0] * n[0], (c[0] + 1) * n[0]))


@pytest.mark.parametrize("name,make,pgrid", CASES, ids=[c[0] for c in CASES])
def test_sharded_equals_unsharded_bit_for_bit(name, make, pgrid):
    from paper_2007_05218_b200 import sharded as S
    from paper_2007_05218_b200.binding import Hydro
    wl = make()
    U0 = W.initial_state(wl)
    G0 = W.gather_valid(wl, U0)
    ref = Hydro(wl.params)
    ref.upload(U0, 0)
    sh = S.LocalShards(wl.params, pgrid)
    for r, sl in shard_blocks(wl, pgrid):
        s = sh.shards[r]
        wloc = W.Workload("shard", wl.kind, s.params, 1, seed=wl.seed, extra=wl.extra)
        s.h.upload(W.scatter_valid(wloc, np.ascontiguousarray(G0[sl]), ghost_value=np.nan), 0)
        s.wl = wloc
    # ghost zones after one sharded fill = the unsharded fill's (every zone of every box, corners included)
    ref.hydro_fill_ghosts(0)
    sh.fill(0)
    Ur = ref.download(0).reshape(wl.state_shape)
    from paper_2007_05218_b200.sharded import proc_coords
    for s in sh.shards:
        Us = s.h.download(0).reshape(s.wl.state_shape)
        c = proc_coords(s.rank, pgrid)
        for b in range(s.wl.nboxes):
            lb = (b % s.wl.NB[0], (b // s.wl.NB[0]) % s.wl.NB[1], b // (s.wl.NB[0] * s.wl.NB[1]))
            gb = [c[d] * s.wl.NB[d] + lb[d] for d in range(3)]
            assert np.array_equal(Us[b], Ur[(gb[2] * wl.NB[1] + gb[1]) * wl.NB[0] + gb[0]]), (s.rank, b)
    # three steps: same dt, same valid zones, bit for bit
    for _ in range(3):
        assert sh.step() == ref.step_explicit()
    Gr = W.gather_valid(wl, ref.download(0).reshape(U0.shape))
    for r, sl in shard_blocks(wl, pgrid):
        s = sh.shards[r]
        assert np.array_equal(W.gather_valid(s.wl, s.h.download(0).reshape(s.wl.state_shape)), Gr[sl]), r
    tr, ts = np.array(ref.hydro_conserved_totals(0)), np.array(sh.totals())
    scale = np.abs(Gr).sum(axis=(1, 2, 3))[[0, 1, 2, 3, 4] + list(range(6, wl.nvar))] * np.prod(wl.dx)
    assert np.all(np.abs(tr - ts) <= 1e-13 * scale)
    # and the loop is closed to the oracle, not only to the unsharded CUDA run: the state gathered from the shards
    # against three oracle steps of the unsharded domain (north_star's multi-step bound)
    from oracle import oracle_binding as O
    from parity_util import rel_err
    p = O.make_params(wl.params)
    Uo, U1 = U0.copy(), np.zeros_like(U0)
    for _ in range(3):
        O.step(p, Uo, U1)
    Gs = np.empty_like(Gr)
    for r, sl in shard_blocks(wl, pgrid):
        s = sh.shards[r]
        Gs[sl] = W.gather_valid(s.wl, s.h.download(0).reshape(s.wl.state_shape))
    e = rel_err(wl, W.scatter_valid(wl, Gs, ghost_value=np.nan), Uo)
    assert np.all(e <= 1e-10), e


def test_a_shard_refuses_hydro_step_and_reports_halo_sizes():
    from paper_2007_05218_b200 import binding as B
    from paper_2007_05218_b200 import sharded as S
    wl = W.config(5, ndom=(64, 32, 32), nbox=(16, 16, 16), nspec=3)
    s = S.Shard(wl.params, (2, 1, 1), 0)
    with pytest.raises(B.HydroError) as ei:
        s.h.hydro_step(1)
    assert ei.value.code == B.HYDRO_EINVAL
    p = B.make_params(s.params)
    nt = [16 + 8] * 3
    # x halo: 2x2 face boxes (y, z), 9 components, 4 layers, full padded y and z extent
    assert B.hydro_halo_bytes(p, 0) == 9 * 4 * nt[1] * nt[2] * 2 * 2 * 8
    assert B.hydro_halo_bytes(p, 2) == 9 * 4 * nt[0] * nt[1] * 2 * 2 * 8 and B.hydro_halo_bytes(p, 3) == 0


def _dist_rank(rank, world, port, pgrid, q):
    """one process per shard, all on cuda:0, gloo transport: the ShardedHydro driver end to end"""
    import os
    import torch.distributed as dist
    from paper_2007_05218_b200 import sharded as S
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = W.config(5, ndom=(64, 32, 64), nbox=(16, 16, 16), nspec=3)
    G0 = W.gather_valid(wl, W.initial_state(wl))
    sh = S.ShardedHydro(wl.params, pgrid, "cuda:0")
    sl = dict(shard_blocks(wl, pgrid))[rank]
    wloc = W.Workload("shard", wl.kind, sh.shard.params, 1, seed=wl.seed, extra=wl.extra)
    sh.shard.h.upload(W.scatter_valid(wloc, np.ascontiguousarray(G0[sl]), ghost_value=np.nan), 0)
    dts = [sh.step() for _ in range(2)]
    tot = sh.totals()
    q.put((rank, dts, tot, W.gather_valid(wloc, sh.shard.h.download(0).reshape(wloc.state_shape))))
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_driver_over_two_processes_on_one_gpu():
    """ShardedHydro (one process per shard, torch.distributed point-to-point halo exchange, allreduce of dt and
    totals) with the gloo transport and both processes on cuda:0: the processes never wait on each other's
    kernels, only on the host-side exchange.  Same dt and bit-identical valid zones as the unsharded run."""
    import os
    import torch.multiprocessing as mp
    from paper_2007_05218_b200.binding import Hydro
    pgrid = (2, 1, 1)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33000 + os.getpid() % 2000
    procs = [ctx.Process(target=_dist_rank, args=(r, 2, port, pgrid, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    wl = W.config(5, ndom=(64, 32, 64), nbox=(16, 16, 16), nspec=3)
    U0 = W.initial_state(wl)
    ref = Hydro(wl.params)
    ref.upload(U0, 0)
    dts = [ref.step_explicit() for _ in range(2)]
    Gr = W.gather_valid(wl, ref.download(0).reshape(U0.shape))
    blocks = dict(shard_blocks(wl, pgrid))
    for rank, dts_r, tot, G in res:
        assert dts_r == dts
        assert np.array_equal(G, Gr[blocks[rank]]), rank
    assert res[0][2] == res[1][2]                                  # the allreduced totals agree on both ranks

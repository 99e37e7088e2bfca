"""GPU parity of the two-level ghost fill O13 (hydro_fill_from_coarse, csrc/amr_fill.cuh) against
oracle_fill_from_coarse: the same zones written (everything else untouched), values equal to rounding (the
default build contracts slope*xi + value into FMAs; with the dyadic linear field bit for bit), and one RK2 step
of a refined patch inside a coarse level, ghost zones from the coarse level at both stages, against the oracle."""
import numpy as np
import pytest

from oracle import oracle_binding as O
from paper_2007_05218_b200 import workloads as W
from test_oracle_amr import EXT, coarse_field, levels

pytestmark = pytest.mark.gpu

CASES = [
    dict(ratio=2, lo=(4, 4, 4), patch=(8, 8, 8), nbox_f=(8, 16, 8), nbox_c=(8, 8, 8)),
    dict(ratio=4, lo=(3, 5, 2), patch=(6, 4, 8), nbox_f=(12, 16, 16), nbox_c=(16, 8, 8)),
    dict(ratio=2, lo=(4, 0, 0), patch=(8, 16, 6), nbox_f=(16, 16, 12), nbox_c=(8, 16, 8), bc_c=(W.OUTFLOW, W.PERIODIC, W.REFLECT)),
]


def hydro(wl):
    from paper_2007_05218_b200.binding import Hydro
    return Hydro(wl.params)


@pytest.mark.parametrize("case", CASES)
def test_fill_from_coarse_matches_oracle(case):
    wc, wf = levels(ndom_c=(16, 16, 16), nspec=2, **case)
    rng = np.random.default_rng(11)
    Uc = W.scatter_valid(wc, rng.standard_normal((wc.nvar, 16, 16, 16)), ghost_value=np.nan)
    nf = wf.params["ndom"]
    Uf = W.scatter_valid(wf, rng.standard_normal((wf.nvar, nf[2], nf[1], nf[0])), ghost_value=np.nan)
    pc, pf = O.make_params(wc.params), O.make_params(wf.params)
    hc, hf = hydro(wc), hydro(wf)
    hc.upload(Uc, 0); hf.upload(Uf, 1)
    hc.hydro_fill_ghosts(0); hf.hydro_fill_ghosts(1)
    hf.hydro_fill_from_coarse(1, hc, 0, case["lo"], case["ratio"])
    O.fill_ghosts(pc, Uc); O.fill_ghosts(pf, Uf)
    O.fill_from_coarse(pf, Uf, pc, Uc, case["lo"], case["ratio"])
    G = hf.download(1).reshape(Uf.shape)
    assert np.array_equal(np.isnan(G), np.isnan(Uf))
    assert not np.isnan(G).any()                                     # fine-fine, physical and coarse-fine fills cover every ghost
    assert np.allclose(G, Uf, rtol=1e-15, atol=1e-15)


def test_linear_field_bit_for_bit_and_errors():
    from paper_2007_05218_b200 import binding as B
    wc, wf = levels(ratio=4, bc_c=W.OUTFLOW, lo=(4, 4, 4), patch=(8, 8, 8))
    f = lambda c, x, y, z: (1 + c) * 0.5 + 2.0 * x - 0.75 * y + 1.25 * z * (1 + c % 3)
    Uc = coarse_field(wc, f)
    Uf = np.full(wf.state_shape, np.nan).reshape(-1)
    hc, hf = hydro(wc), hydro(wf)
    hc.upload(Uc, 0); hf.upload(Uf, 0)
    hf.hydro_fill_from_coarse(0, hc, 0, (4, 4, 4), 4)
    O.fill_from_coarse(O.make_params(wf.params), Uf, O.make_params(wc.params), Uc, (4, 4, 4), 4)
    assert np.array_equal(hf.download(0), Uf, equal_nan=True)
    for lo, ratio in (((4, 4, 4), 3), ((12, 4, 4), 4)):
        with pytest.raises(B.HydroError) as ei:
            hf.hydro_fill_from_coarse(0, hc, 0, lo, ratio)
        assert ei.value.code == B.HYDRO_EINVAL


def test_one_rk2_step_of_a_refined_patch_inside_a_coarse_level():
    """Coarse 32^3 (config-3 recipe) with its central 16^3 refined by 2 (a 32^3 patch in 16^3 boxes): both levels take
    one RK2 step with the same dt, the patch's outer ghost zones interpolated from the coarse level at both stages
    (no averaging down, no refluxing: the ghost fill is the row built)."""
    wc = W.config(3, ndom=(32, 32, 32), nbox=(16, 16, 16), nspec=2)
    lo, ratio = (8, 8, 8), 2
    wf = W.config(3, ndom=(32, 32, 32), nbox=(16, 16, 16), nspec=2)
    dx = wc.dx
    wf.params["prob_lo"] = [lo[d] * dx[d] for d in range(3)]
    wf.params["prob_hi"] = [(lo[d] + 16) * dx[d] for d in range(3)]
    wf.params["bc_lo"] = [EXT] * 3
    wf.params["bc_hi"] = [EXT] * 3
    Uc0 = W.initial_state(wc)
    # the fine initial state: the coarse recipe's smooth part sampled... simply the interpolated coarse data, via the oracle:
    # a fine patch whose valid zones are piecewise-constant children of the coarse zones (conservative), ghosts NaN
    Gc = W.gather_valid(wc, Uc0)
    Gf = np.repeat(np.repeat(np.repeat(Gc[:, 8:24, 8:24, 8:24], 2, axis=1), 2, axis=2), 2, axis=3)
    Uf0 = W.scatter_valid(wf, Gf, ghost_value=np.nan)
    pc, pf = O.make_params(wc.params), O.make_params(wf.params)
    hc, hf = hydro(wc), hydro(wf)
    hc.upload(Uc0, 0); hf.upload(Uf0, 0)
    dt = min(hc.hydro_estimate_dt(), hf.hydro_estimate_dt())
    dt_o = min(O.estimate_dt(pc, Uc0), O.estimate_dt(pf, Uf0))
    assert abs(dt - dt_o) <= 1e-14 * dt_o
    Uc, Uc1, Uf, Uf1 = Uc0.copy(), np.zeros_like(Uc0), Uf0.copy(), np.zeros_like(Uf0)
    for stage in (0, 1):
        hc.hydro_fill_ghosts(stage); hf.hydro_fill_ghosts(stage)
        hf.hydro_fill_from_coarse(stage, hc, stage, lo, ratio)
        hc.hydro_advance_stage(stage, dt_o); hf.hydro_advance_stage(stage, dt_o)
        src_c, src_f = (Uc, Uf) if stage == 0 else (Uc1, Uf1)
        O.fill_ghosts(pc, src_c); O.fill_ghosts(pf, src_f)
        O.fill_from_coarse(pf, src_f, pc, src_c, lo, ratio)
        O.advance_stage(pc, stage, dt_o, Uc, Uc1); O.advance_stage(pf, stage, dt_o, Uf, Uf1)
    from parity_util import rel_err
    assert np.all(rel_err(wc, hc.download(0).reshape(Uc.shape), Uc) <= 1e-12)
    e = rel_err(wf, hf.download(0).reshape(Uf.shape), Uf)
    assert np.all(e <= 1e-12), e
    assert np.abs(W.gather_valid(wf, Uf) - Gf).max() > 1e-4          # the patch did evolve


@pytest.mark.parametrize("ratio", [2, 4])
def test_average_down_bit_for_bit(ratio):
    wc, wf = levels(ratio=ratio, lo=(4, 2, 6), patch=(8, 4, 6), nbox_c=(8, 16, 8), nspec=2)
    wf.params["nbox"] = [wf.params["ndom"][0] // 2, wf.params["ndom"][1], wf.params["ndom"][2] // 2]
    rng = np.random.default_rng(21)
    nf = wf.params["ndom"]
    Uf = W.scatter_valid(wf, rng.standard_normal((wf.nvar, nf[2], nf[1], nf[0])), ghost_value=np.nan)
    Uc = W.scatter_valid(wc, rng.standard_normal((wc.nvar, 16, 16, 16)), ghost_value=np.nan)
    hc, hf = hydro(wc), hydro(wf)
    hc.upload(Uc, 1); hf.upload(Uf, 0)
    hc.hydro_average_down(1, hf, 0, (4, 2, 6), ratio)
    O.average_down(O.make_params(wc.params), Uc, O.make_params(wf.params), Uf, (4, 2, 6), ratio)
    assert np.array_equal(hc.download(1).reshape(Uc.shape), Uc, equal_nan=True)


def test_two_level_driver_three_steps_against_the_oracle():
    """paper_2007_05218_b200/amr.py: three RK2 steps of a coarse level with a 2x-refined patch on its reflecting
    floor (config-4 recipe: gravity, 2 species), fill_from_coarse at both stages and average_down after every
    step, against the same sequence of oracle calls."""
    from paper_2007_05218_b200 import amr
    from parity_util import rel_err
    wc = W.config(4, ndom=(32, 32, 32), nbox=(16, 16, 16), nspec=2)
    lo, extent, ratio = (8, 8, 0), (16, 16, 8), 2
    tl = amr.TwoLevelHydro(wc.params, lo, extent, ratio, (16, 16, 16))
    assert tl.fine_params["bc_lo"] == [EXT, EXT, W.REFLECT] and tl.fine_params["bc_hi"] == [EXT, EXT, EXT]
    wf = W.Workload("patch", wc.kind, tl.fine_params, 1, seed=wc.seed, extra=wc.extra)
    Uc = W.initial_state(wc)
    Gc = W.gather_valid(wc, Uc)
    Gf = np.repeat(np.repeat(np.repeat(Gc[:, 0:8, 8:24, 8:24], 2, axis=1), 2, axis=2), 2, axis=3)
    Uf = W.scatter_valid(wf, Gf, ghost_value=np.nan)
    tl.coarse.upload(Uc, 0); tl.fine.upload(Uf, 0)
    pc, pf = O.make_params(wc.params), O.make_params(tl.fine_params)
    Uc1, Uf1 = np.zeros_like(Uc), np.zeros_like(Uf)
    for _ in range(3):
        dt_o = min(O.estimate_dt(pc, Uc), O.estimate_dt(pf, Uf))
        for stage in (0, 1):
            sc, sf = (Uc, Uf) if stage == 0 else (Uc1, Uf1)
            O.fill_ghosts(pc, sc); O.fill_ghosts(pf, sf)
            O.fill_from_coarse(pf, sf, pc, sc, lo, ratio)
            O.advance_stage(pc, stage, dt_o, Uc, Uc1); O.advance_stage(pf, stage, dt_o, Uf, Uf1)
        O.average_down(pc, Uc, pf, Uf, lo, ratio)
        dt = tl.step()
        assert abs(dt - dt_o) <= 1e-12 * dt_o
    assert np.all(rel_err(wc, tl.coarse.download(0).reshape(Uc.shape), Uc) <= 1e-11)
    assert np.all(rel_err(wf, tl.fine.download(0).reshape(Uf.shape), Uf) <= 1e-11)
    # the coarse zones under the patch are the means of their children
    Gc2, Gf2 = W.gather_valid(wc, Uc), W.gather_valid(wf, Uf)
    kids = Gf2.reshape(wf.nvar, 8, 2, 16, 2, 16, 2).mean(axis=(2, 4, 6))
    assert np.allclose(Gc2[:, 0:8, 8:24, 8:24], kids, rtol=1e-14, atol=1e-15)

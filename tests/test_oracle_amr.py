"""Pins of the oracle's two-level ghost fill O13 (oracle_fill_from_coarse; readings A1-A5 in oracle/hydro_oracle.c):
what the mathematics fixes about a conservative linear interpolation from a coarse level into the ghost zones of
a refined patch.  Nothing here comes from the CUDA path."""
import copy

import numpy as np
import pytest

from oracle import oracle_binding as O
from paper_2007_05218_b200 import workloads as W

EXT = 3


def levels(ndom_c=(16, 16, 16), nbox_c=(8, 8, 8), lo=(4, 4, 4), patch=(8, 8, 8), ratio=2, nbox_f=None, nspec=1,
           bc_c=W.PERIODIC):
    """coarse workload + the fine patch [lo, lo+patch) refined by ratio (its interior faces EXTERNAL)"""
    wc = W.uniform(ndom_c, nbox_c, nspec, (1, 0, 0, 0, 1), bc=bc_c)
    wf = copy.deepcopy(wc)
    p = wf.params
    dx = wc.dx
    p["ndom"] = [ratio * n for n in patch]
    p["nbox"] = list(nbox_f or p["ndom"])
    p["prob_lo"] = [wc.params["prob_lo"][d] + lo[d] * dx[d] for d in range(3)]
    p["prob_hi"] = [wc.params["prob_lo"][d] + (lo[d] + patch[d]) * dx[d] for d in range(3)]
    for d in range(3):
        p["bc_lo"][d] = wc.params["bc_lo"][d] if (lo[d] == 0 and wc.params["bc_lo"][d] != W.PERIODIC) else EXT
        p["bc_hi"][d] = wc.params["bc_hi"][d] if (lo[d] + patch[d] == ndom_c[d] and wc.params["bc_hi"][d] != W.PERIODIC) else EXT
    return wc, wf


def coarse_field(wc, f):
    """coarse state whose component c at zone centre (x, y, z) is f(c, x, y, z); ghosts by the coarse BCs"""
    n = wc.params["ndom"]
    x = [(np.arange(n[d]) + 0.5) * wc.dx[d] + wc.params["prob_lo"][d] for d in range(3)]
    G = np.stack([f(c, x[0][None, None, :], x[1][None, :, None], x[2][:, None, None]) * np.ones((n[2], n[1], n[0]))
                  for c in range(wc.nvar)])
    U = W.scatter_valid(wc, G, ghost_value=np.nan)
    O.fill_ghosts(O.make_params(wc.params), U)
    return U


def fine_centres(wf):
    """(x, y, z) arrays of the zone centres of the padded fine box 0 (single-box patches)"""
    ng, nt = wf.ng, wf.nt
    return [(np.arange(nt[d]) - ng + 0.5) * wf.dx[d] + wf.params["prob_lo"][d] for d in range(3)]


def ghost_mask_external(wf):
    """padded-zone mask (single box): index across an EXTERNAL face in at least one dimension (reading A5)"""
    ng, nt, nd = wf.ng, wf.nt, wf.params["ndom"]
    m = np.zeros((nt[2], nt[1], nt[0]), bool)
    for d, ax in ((0, 2), (1, 1), (2, 0)):
        g = np.arange(nt[d]) - ng
        out = ((g < 0) & (wf.params["bc_lo"][d] == EXT)) | ((g >= nd[d]) & (wf.params["bc_hi"][d] == EXT))
        sh = [1, 1, 1]
        sh[ax] = nt[d]
        m |= out.reshape(sh)
    return m


@pytest.mark.parametrize("ratio", [2, 4])
def test_linear_data_is_reproduced_bit_for_bit(ratio):
    """A linear field with dyadic coefficients on a dyadic grid: every slope, product and sum is exact, the limiter
    is inactive (dp == dm), so every filled ghost zone holds the field's value at its own centre, bit for bit."""
    wc, wf = levels(ratio=ratio, bc_c=W.OUTFLOW, lo=(4, 4, 4), patch=(8, 8, 8))
    f = lambda c, x, y, z: (1 + c) * 0.5 + 2.0 * x - 0.75 * y + 1.25 * z * (1 + c % 3)
    Uc = coarse_field(wc, f)
    Uf = np.full(wf.state_shape, np.nan).reshape(-1)
    O.fill_from_coarse(O.make_params(wf.params), Uf, O.make_params(wc.params), Uc, (4, 4, 4), ratio)
    Uf = Uf.reshape(wf.state_shape)[0]
    xs = fine_centres(wf)
    m = ghost_mask_external(wf)
    assert m.sum() == np.prod(wf.nt) - np.prod(wf.nb)                # all six faces are interior: every ghost zone
    for c in range(wf.nvar):
        exact = f(c, xs[0][None, None, :], xs[1][None, :, None], xs[2][:, None, None])
        assert np.array_equal(Uf[c][m], exact[m]), c
        assert np.all(np.isnan(Uf[c][~m]))                           # ... and no other zone is touched


def test_children_average_to_the_parent_and_extrema_stay_flat():
    wc, wf = levels(ratio=2, lo=(4, 4, 4), patch=(8, 8, 8))
    rng = np.random.default_rng(3)
    G = rng.standard_normal((wc.nvar, 16, 16, 16))
    G[0, 2, 5, 3] = 50.0                                             # a strict local extremum of component 0
    Uc = W.scatter_valid(wc, G, ghost_value=np.nan)
    pc = O.make_params(wc.params)
    O.fill_ghosts(pc, Uc)
    Uf = np.full(wf.state_shape, np.nan).reshape(-1)
    O.fill_from_coarse(O.make_params(wf.params), Uf, pc, Uc, (4, 4, 4), 2)
    Uf = Uf.reshape(wf.state_shape)[0]
    ng = wf.ng
    # the 2 x 2 x 2 children of coarse zone (3, 5, 2) are fine zones (-2..-1, 2..3, -4..-3): all ghosts of the patch
    kids = Uf[:, ng - 4:ng - 2, ng + 2:ng + 4, ng - 2:ng]
    assert np.all(kids[0] == 50.0)                                   # extremum: all three limited slopes vanish
    for c in range(1, wf.nvar):
        assert kids[c].mean() == pytest.approx(G[c, 2, 5, 3], rel=1e-14, abs=1e-15)
    # monotone: every child lies within the range of the parent's 27 neighbours (here: of the 7-point stencil per dimension)
    for c in range(wf.nvar):
        nb = G[c, 1:4, 4:7, 2:5]
        assert kids[c].min() >= nb.min() - 1e-14 and kids[c].max() <= nb.max() + 1e-14


def test_patch_on_a_wall_uses_the_coarse_boundary_condition_in_the_corner():
    """The patch sits on the reflecting low-z wall of the coarse domain: its low-z ghosts are O1's (reflect), its
    x and y faces are EXTERNAL; the corner ghost zones (x outside, z below the wall) come from the coarse level's
    own ghost zones, i.e. mirrored data with rho*w negated (reading A4)."""
    wc, wf = levels(ndom_c=(16, 16, 16), nbox_c=(8, 16, 8), lo=(4, 4, 0), patch=(8, 8, 4), ratio=2,
                    bc_c=(W.PERIODIC, W.PERIODIC, W.REFLECT))
    assert wf.params["bc_lo"] == [EXT, EXT, W.REFLECT] and wf.params["bc_hi"] == [EXT, EXT, EXT]
    f = lambda c, x, y, z: (2.0 + c) + 0.5 * np.sin(2 * np.pi * x) * (z + 0.25) + (0.3 * z if c == W.MZ else 0.0)
    Uc = coarse_field(wc, f)
    pf = O.make_params(wf.params)
    Uf = np.full(wf.state_shape, np.nan).reshape(-1)
    O.fill_from_coarse(pf, Uf, O.make_params(wc.params), Uc, (4, 4, 0), 2)
    Uf = Uf.reshape(wf.state_shape)[0]
    ng = wf.ng
    m = ghost_mask_external(wf)
    assert np.all(np.isfinite(Uf[:, m])) and np.all(np.isnan(Uf[:, ~m]))
    # corner column: fine ghost (i = -1, j = 3, k = -1) mirrors (i = -1, j = 3, k = 0) with rho*w negated
    lo_k, up_k = Uf[:, ng - 1, ng + 3, ng - 1], Uf[:, ng, ng + 3, ng - 1]
    for c in range(wf.nvar):
        assert lo_k[c] == pytest.approx(-up_k[c] if c == W.MZ else up_k[c], rel=1e-14)


def test_fill_ghosts_leaves_external_faces_alone_and_rejects_bad_patches():
    wc, wf = levels(ratio=2, lo=(4, 4, 4), patch=(8, 8, 8), nbox_f=(8, 16, 8))
    rng = np.random.default_rng(5)
    U = W.scatter_valid(wf, rng.standard_normal((wf.nvar, 16, 16, 16)), ghost_value=np.nan)
    pf = O.make_params(wf.params)
    O.fill_ghosts(pf, U)
    Ub = U.reshape(wf.state_shape)
    ng = wf.ng
    # box 0 of the 2 x 1 x 2 boxes: its high-x ghosts are the neighbour box's valid zones, its low-x ghosts stay NaN
    assert np.all(np.isnan(Ub[0, :, ng:-ng, ng:-ng, :ng])) and np.all(np.isfinite(Ub[0, :, ng:-ng, ng:-ng, -ng:]))
    Uc = coarse_field(wc, lambda c, x, y, z: 1.0 + x)
    pc = O.make_params(wc.params)
    with pytest.raises(RuntimeError):
        O.fill_from_coarse(pf, U, pc, Uc, (4, 4, 4), 3)                      # ratio must be 2 or 4
    with pytest.raises(RuntimeError):
        O.fill_from_coarse(pf, U, pc, Uc, (12, 4, 4), 2)                     # the patch sticks out of the coarse domain


@pytest.mark.parametrize("ratio", [2, 4])
def test_average_down_is_exact_for_linear_data_and_conserves(ratio):
    wc, wf = levels(ratio=ratio, bc_c=W.OUTFLOW, lo=(4, 2, 6), patch=(8, 4, 6), nbox_f=None)
    wf.params["nbox"] = [wf.params["ndom"][0] // 2, wf.params["ndom"][1], wf.params["ndom"][2] // 2]     # 2 x 1 x 2 fine boxes
    pc, pf = O.make_params(wc.params), O.make_params(wf.params)
    # fine data = a dyadic linear field at the fine centres: the mean of the children is the field at the parent centre
    f = lambda c, x, y, z: (1 + c) * 0.25 + 2.0 * x - 0.75 * y + 1.5 * z
    nf = wf.params["ndom"]
    xs = [(np.arange(nf[d]) + 0.5) * wf.dx[d] + wf.params["prob_lo"][d] for d in range(3)]
    Gf = np.stack([f(c, xs[0][None, None, :], xs[1][None, :, None], xs[2][:, None, None]) * np.ones((nf[2], nf[1], nf[0]))
                   for c in range(wf.nvar)])
    Uf = W.scatter_valid(wf, Gf, ghost_value=np.nan)
    Uc = W.scatter_valid(wc, np.full((wc.nvar, 16, 16, 16), -7.0), ghost_value=np.nan)
    O.average_down(pc, Uc, pf, Uf, (4, 2, 6), ratio)
    Gc = W.gather_valid(wc, Uc)
    xc = [(np.arange(16) + 0.5) * wc.dx[d] for d in range(3)]
    exact = np.stack([f(c, xc[0][None, None, :], xc[1][None, :, None], xc[2][:, None, None]) * np.ones((16, 16, 16))
                      for c in range(wc.nvar)])
    patch = (slice(None), slice(6, 12), slice(2, 6), slice(4, 12))
    assert np.array_equal(Gc[patch], exact[patch])
    outside = np.ones((16, 16, 16), bool)
    outside[patch[1:]] = False
    assert np.all(Gc[:, outside] == -7.0)                               # nothing outside the patch is touched
    # conservation with random fine data: coarse total over the patch == fine total
    rng = np.random.default_rng(9)
    Gr = rng.standard_normal(Gf.shape)
    Uf = W.scatter_valid(wf, Gr, ghost_value=np.nan)
    O.average_down(pc, Uc, pf, Uf, (4, 2, 6), ratio)
    Gc = W.gather_valid(wc, Uc)
    for c in range(wc.nvar):
        assert Gc[c][patch[1:]].sum() * np.prod(wc.dx) == pytest.approx(Gr[c].sum() * np.prod(wf.dx), rel=1e-13, abs=1e-15)

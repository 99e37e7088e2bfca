"""Pins of the optional shock flattening O10: worked line
examples computed by hand from the formula, the exact no-op property on shock-free flow, conservation,
and the Sod solution.  Nothing here comes from the CUDA path."""
import copy

import numpy as np

from oracle import oracle_binding as O
from paper_2007_05218_b200 import workloads as W
from test_oracle_scheme import exact_riemann_sod, run_steps, run_to


def test_flatten_line_strong_compressive_jump():
    # p jumps 1 -> 10 between zones 5 and 6, flow converging: |dp|/|dp2| = 1 -> z = 1, chi = 1 at zones
    # 5 and 6 (each also sees the other as its low-pressure-side neighbour); zones 4 and 7 have dp = 0:
    # no neighbour is consulted, they keep their parabolas
    pr = np.array([1, 1, 1, 1, 1, 1, 10, 10, 10, 10, 10, 10], float)
    un = np.array([1.0] * 6 + [0.0] * 6)
    assert np.array_equal(O.flatten_line(pr, un), [1, 1, 1, 1, 1, 0, 0, 1, 1, 1, 1, 1])
    # mirror image of the line (pressure and velocity reversed, velocity sign flipped): mirrored result
    assert np.array_equal(O.flatten_line(pr[::-1].copy(), -un[::-1].copy()), [1, 1, 1, 1, 1, 0, 0, 1, 1, 1, 1, 1])
    # a three-zone ramp 1, 4, 10: the zone below the ramp (dp > 0 towards it) is flattened through its
    # low-pressure-side rule only if ITS neighbour on that side is a shock zone -- here zone 4 looks at 3
    pr2 = np.array([1, 1, 1, 1, 1, 4, 10, 10, 10, 10, 10, 10], float)
    f2 = O.flatten_line(pr2, un)
    m2 = O.flatten_line(pr2[::-1].copy(), -un[::-1].copy())
    assert np.array_equal(f2, m2[::-1])
    # the same jump in an expanding flow (un increasing) is not a shock
    assert np.array_equal(O.flatten_line(pr, un[::-1].copy()), np.ones(12))


def test_flatten_line_ramp_value_exact():
    # zone 5: dp = p6 - p4 = 13, dp2 = p7 - p3 = 16, zeta = 13/16 -> z = 10*(0.8125 - 0.75) = 0.625 exactly
    pr = np.array([1, 1, 1, 1, 2, 8, 15, 17, 17, 17, 17, 17], float)
    un = np.array([1.0] * 6 + [0.0] * 6)
    f = O.flatten_line(pr, un)
    # zone 6: dp = 9, dp2 = p8 - p4 = 15 -> zeta = 0.6 -> z = 0; zone 4: dp = 7, dp2 = 14 -> zeta 0.5 -> z = 0
    assert f[5] == 1.0 - 0.625
    assert f[4] == 1.0 and f[7] == 1.0 and f[3] == 1.0
    # zone 6 has dp > 0, so it looks at zone 5 (s = +1, i - s = 5): flattened by the same 0.625
    assert f[6] == 1.0 - 0.625


def test_flatten_line_weak_jump_untouched():
    pr = np.array([1.0] * 6 + [1.3] * 6)        # |dp| / min p = 0.3 <= 0.33
    un = np.array([1.0] * 6 + [0.0] * 6)
    assert np.array_equal(O.flatten_line(pr, un), np.ones(12))


def test_flatten_is_exact_noop_without_shocks():
    # config-3 recipe: p = 1 everywhere -> dp = 0 -> z = 0 -> coefficient 1 -> 1*aL + 0*a == aL exactly
    wl = W.config(3, ndom=(32, 16, 16), nbox=(16, 8, 8), nspec=2)
    U0 = W.initial_state(wl)
    A, B = U0.copy(), U0.copy()
    run_steps(wl, A, 2)
    wf = copy.deepcopy(wl); wf.params["flatten"] = 1
    run_steps(wf, B, 2)
    assert np.array_equal(A, B)


def test_flatten_needs_four_ghost_zones():
    wl = W.config(3, ndom=(16, 16, 16), nbox=(16, 16, 16), nspec=0)
    wl.params["ng"] = 3; wl.params["flatten"] = 1
    assert O.state_doubles(O.make_params(wl.params)) == 0


def test_flatten_sod_conserves_and_still_converges():
    errs = {}
    for N in (64, 128):
        wl = W.config(1, ndom=(N, 4, 4)); wl.params["flatten"] = 1
        U0 = W.initial_state(wl)
        p = O.make_params(wl.params)
        t0 = O.conserved_totals(p, U0)
        run_to(wl, U0, 0.2)
        G = W.gather_valid(wl, U0)
        sample, st = exact_riemann_sod()
        sub = (np.arange(64) + 0.5) / 64
        xf = (np.arange(N)[:, None] + sub[None, :]) / N
        exact = sample((xf - 0.5) / 0.2).mean(axis=1)
        errs[N] = np.abs(G[0, 0, 0] - exact).mean()
        assert np.abs(G[W.MY]).max() == 0.0
        # mass: outflow boundaries are still undisturbed at t = 0.2, so totals are conserved to rounding
        t1 = O.conserved_totals(p, U0)
        assert abs(t1[0] - t0[0]) <= 1e-13 * abs(t0[0])
        # no overshoot behind the shock: density stays within the exact solution's range
        assert G[0].max() <= 1.0 + 1e-12 and G[0].min() >= 0.125 - 1e-12
    assert errs[64] > errs[128] and errs[64] / errs[128] >= 1.5
    assert errs[128] < 6e-3


def test_flatten_box_decomposition_invariance_bitwise():
    wl = W.config(2, ndom=(32, 32, 32), nbox=(32, 32, 32)); wl.params["flatten"] = 1
    G0 = W.gather_valid(wl, W.initial_state(wl))
    out = []
    for nbox in [(32, 32, 32), (16, 16, 16), (8, 16, 32)]:
        w = W.with_boxes(wl, nbox)
        U = W.scatter_valid(w, G0)
        run_steps(w, U, 3)
        out.append(W.gather_valid(w, U))
    assert np.array_equal(out[0], out[1]) and np.array_equal(out[0], out[2])
    # the blast is a strong shock: flattening must have changed the solution
    w0 = copy.deepcopy(wl); w0.params["flatten"] = 0
    U = W.scatter_valid(w0, G0)
    run_steps(w0, U, 3)
    assert not np.array_equal(out[0], W.gather_valid(w0, U))


def test_flatten_keeps_the_blast_mirror_symmetric():
    # a point blast centred on a zone corner has mirror pairs of zones; the dp == 0 rule (reading F3) is
    # what keeps O10 from preferring one direction
    wl = W.config(2, ndom=(32, 32, 32), nbox=(16, 16, 32)); wl.params["flatten"] = 1
    U = W.initial_state(wl)
    run_steps(wl, U, 12)
    rho = W.gather_valid(wl, U)[0]
    assert np.allclose(rho, rho[::-1, ::-1, ::-1], rtol=1e-12, atol=0)
    assert rho.max() > 1.5                      # the shock has formed and moved

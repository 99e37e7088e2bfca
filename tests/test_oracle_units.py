"""Pins of the oracle's unit steps against what the mathematics fixes (SURVEY.md 8(c)
P5, P6, P11, P12).  Expected values are exact rationals / closed forms worked out from
the cited definitions (CW84 eqs. 1.6-1.10; Toro HLLC with Davis speeds), never produced
by the oracle or the CUDA path."""
from fractions import Fraction as Fr

import numpy as np
import pytest

import golden_util
from oracle import oracle_binding as O
from paper_2007_05218_b200 import workloads as W


# ---------------------------------------------------------------- O2 primitives
def test_cons_to_prim_gamma_law():
    # rho=2, u=(1,-2,3), p=0.8 with gamma=1.4: rho*e = p/(gamma-1) = 2
    Uc = np.array([2.0, 2.0, -4.0, 6.0, 2.0 + 0.5 * 2.0 * 14.0, 2.0, 0.5, 1.5])
    q = O.cons_to_prim(1.4, 1e-12, 1e-14, 2, Uc)
    assert q[0] == 2.0 and q[1] == 1.0 and q[2] == -2.0 and q[3] == 3.0
    assert q[4] == pytest.approx(0.8, rel=1e-15)
    assert q[5] == 0.25 and q[6] == 0.75


def test_cons_to_prim_floors():
    q = O.cons_to_prim(1.4, 1e-12, 1e-14, 0, np.array([0.0, 0.0, 0.0, 0.0, 0.0, -1.0]))
    assert q[0] == 1e-12 and q[4] == 1e-14


# ---------------------------------------------------------------- O3/O4 PPM (P5)
def test_ppm_worked_example_exact_rationals():
    # a[-2..3] = 0, 0, 1/10, 1, 2, 3  (line index m = zone + 2)
    a = [Fr(0), Fr(0), Fr(1, 10), Fr(1), Fr(2), Fr(3)]
    s, e, aL, aR = O.ppm_line([float(x) for x in a])
    gold = golden_util.load("ppm_worked.txt")         # exact rationals, SURVEY 8(c) P5
    # slopes (CW 1.7-1.8): s[-1]=0, s[0]=1/5, s[1]=19/20
    assert s[1] == float(gold["s_m1"]) == 0.0
    assert s[2] == pytest.approx(float(gold["s_0"]), rel=2e-16)
    assert s[3] == pytest.approx(float(gold["s_1"]), rel=2e-16)
    # edges (CW 1.6): e[-1/2]=1/60, e[1/2]=17/40, e[3/2]=179/120
    assert e[1] == pytest.approx(float(gold["e_m1half"]), rel=1e-14)
    assert e[2] == pytest.approx(float(gold["e_1half"]), rel=1e-15)
    assert e[3] == pytest.approx(float(gold["e_3half"]), rel=1e-15)
    # zone 0 (m=2): second CW 1.10 branch -> (1/60, 4/15); zone 1 (m=3) untouched
    assert aL[2] == pytest.approx(float(gold["zone0_aL"]), rel=1e-14)
    assert aR[2] == pytest.approx(float(gold["zone0_aR"]), rel=1e-14)
    assert aL[3] == pytest.approx(float(gold["zone1_aL"]), rel=1e-15)
    assert aR[3] == pytest.approx(float(gold["zone1_aR"]), rel=1e-15)
    assert gold["zone0_aR"] == Fr(4, 15) and gold["e_3half"] == Fr(179, 120)


def test_ppm_first_branch_mirror():
    # mirror image of the worked example exercises the other one-sided branch (aL reset)
    a = [3.0, 2.0, 1.0, 0.1, 0.0, 0.0]
    s, e, aL, aR = O.ppm_line(a)
    assert aR[3] == pytest.approx(1.0 / 60.0, rel=1e-14)
    assert aL[3] == pytest.approx(4.0 / 15.0, rel=1e-14)
    assert aL[2] == pytest.approx(179.0 / 120.0, rel=1e-15)
    assert aR[2] == pytest.approx(17.0 / 40.0, rel=1e-15)


def test_ppm_step_is_flat():
    s, e, aL, aR = O.ppm_line([0.0, 0.0, 0.0, 1.0, 1.0, 1.0])
    assert aL[2] == 0.0 and aR[2] == 0.0 and aL[3] == 1.0 and aR[3] == 1.0


def test_ppm_linear_data_exact_midpoints():
    a = 0.5 + 0.25 * np.arange(10)          # exactly representable
    s, e, aL, aR = O.ppm_line(a)
    assert np.all(s[1:-1] == 0.25)
    assert np.all(e[1:-2] == 0.5 * (a[1:-2] + a[2:-1]))
    assert np.all(aL[2:-2] == a[2:-2] - 0.125) and np.all(aR[2:-2] == a[2:-2] + 0.125)


def test_ppm_smooth_fourth_order_edge():
    # limiter inactive (monotone, gently curved): e = 7/12 (a_i + a_i+1) - 1/12 (a_i-1 + a_i+2)
    x = np.arange(12) * 0.1
    a = 1.0 + x + 0.3 * x * x
    s, e, aL, aR = O.ppm_line(a)
    for i in range(1, 9):
        ref = 7.0 / 12.0 * (a[i] + a[i + 1]) - 1.0 / 12.0 * (a[i - 1] + a[i + 2])
        assert e[i] == pytest.approx(ref, rel=1e-14)


def test_ppm_local_extremum_flattened_and_bounds():
    rng = np.random.default_rng(5)
    a = rng.standard_normal(200)
    s, e, aL, aR = O.ppm_line(a)
    for i in range(2, 197):
        lo, hi = min(a[i - 1:i + 2]), max(a[i - 1:i + 2])
        assert lo - 1e-14 <= aL[i] <= hi + 1e-14 and lo - 1e-14 <= aR[i] <= hi + 1e-14
        if (a[i + 1] - a[i]) * (a[i] - a[i - 1]) <= 0:        # extremum -> constant
            assert aL[i] == a[i] and aR[i] == a[i]
        # monotonised parabola has no interior extremum: |aR-aL| >= 6|a - (aL+aR)/2| (CW 1.10)
        d, m = aR[i] - aL[i], a[i] - 0.5 * (aL[i] + aR[i])
        assert abs(d) * (1 + 1e-12) + 1e-15 >= 6.0 * abs(m)


# ---------------------------------------------------------------- O5 HLLC (P6)
SOD_L = [1.0, 0.0, 0.0, 0.0, 1.0, 1.0]
SOD_R = [0.125, 0.0, 0.0, 0.0, 0.1, 0.0]


def test_hllc_sod_interface_worked_example():
    F = O.hllc(0, 1.4, SOD_L, SOD_R)
    cL = np.sqrt(1.4)
    SM = 0.9 / (cL * 1.125)                       # (pR-pL)/(mL-mR), mL=-cL, mR=cL/8
    fac = cL / (cL + SM)                          # rho*_L
    gold = golden_util.load("hllc_worked.txt")
    assert cL == pytest.approx(gold["cL"], rel=1e-15) and np.sqrt(1.4 * 0.1 / 0.125) == pytest.approx(gold["cR"], rel=1e-15)
    assert SM == pytest.approx(gold["SM"], rel=1e-14)
    assert fac == pytest.approx(gold["fac"], rel=1e-14)
    ref = [gold["F_rho"], gold["F_mx"], gold["F_my"], gold["F_mz"], gold["F_E"]]
    assert F[:5] == pytest.approx(ref, rel=1e-14, abs=0)
    assert F[5] == F[0] * 1.0                     # species upwinded from the left (F_rho > 0)
    # independent closed form: F = F_L + S_L (U*_L - U_L), F_L = (0, p, 0, 0, 0)
    assert F[0] == pytest.approx(-cL * (fac - 1.0), rel=1e-14)
    assert F[1] == pytest.approx(1.0 - cL * fac * SM, rel=1e-14)


def test_hllc_stationary_contact_exact():
    for d in range(3):
        F = O.hllc(d, 1.4, [1.0, 0, 0, 0, 1.0, 0.3], [0.125, 0, 0, 0, 1.0, 0.9])
        ref = np.zeros(6); ref[1 + d] = 1.0
        assert np.array_equal(F, ref)             # HLLC keeps the contact (HLL would not)


def test_hllc_consistency_and_supersonic():
    rng = np.random.default_rng(7)
    for _ in range(50):
        q = np.concatenate([[rng.uniform(0.5, 2)], rng.uniform(-1, 1, 3), [rng.uniform(0.5, 2)],
                            rng.uniform(0, 1, 2)])
        for d in range(3):
            r, v, p = q[0], q[1:4], q[4]
            E = p / 0.4 + 0.5 * r * v @ v
            phys = np.array([r * v[d], *(r * v[d] * v + p * np.eye(3)[d]), (E + p) * v[d]])
            assert O.hllc(d, 1.4, q, q)[:5] == pytest.approx(phys, rel=1e-13, abs=1e-14)
    # supersonic to the right: exactly the left physical flux
    qL = np.array([1.0, 5.0, 0.2, -0.1, 1.0, 0.25]); qR = np.array([0.9, 4.8, 0.1, 0.0, 0.8, 0.5])
    r, v, p = qL[0], qL[1:4], qL[4]
    E = p * (1.0 / (1.4 - 1.0)) + 0.5 * r * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2])
    F = O.hllc(0, 1.4, qL, qR)
    assert F[0] == r * v[0] and F[1] == r * v[0] * v[0] + p and F[4] == (E + p) * v[0]
    assert F[5] == F[0] * 0.25
    # supersonic to the left: right flux and right species
    qLm, qRm = qR.copy(), qL.copy(); qLm[1] *= -1; qRm[1] *= -1
    F2 = O.hllc(0, 1.4, qLm, qRm)
    assert F2[0] == -F[0] and F2[1] == F[1] and F2[5] == F2[0] * 0.25


def test_hllc_mirror_symmetry():
    rng = np.random.default_rng(11)
    for _ in range(100):
        qL = np.concatenate([[rng.uniform(0.1, 2)], rng.uniform(-2, 2, 3), [rng.uniform(0.1, 2)], [rng.uniform()]])
        qR = np.concatenate([[rng.uniform(0.1, 2)], rng.uniform(-2, 2, 3), [rng.uniform(0.1, 2)], [rng.uniform()]])
        for d in range(3):
            F = O.hllc(d, 5.0 / 3.0, qL, qR)
            qLm, qRm = qR.copy(), qL.copy()
            qLm[1 + d] *= -1; qRm[1 + d] *= -1
            Fm = O.hllc(d, 5.0 / 3.0, qLm, qRm)
            sign = -np.ones(6); sign[1 + d] = 1.0
            assert Fm == pytest.approx(sign * F, rel=1e-12, abs=1e-13)


def test_hllc_direction_permutation():
    # rotating the velocity components with the direction rotates the momentum fluxes
    qL = np.array([1.0, 0.3, -0.2, 0.5, 1.0, 0.1]); qR = np.array([0.5, -0.1, 0.4, 0.2, 0.6, 0.7])
    Fx = O.hllc(0, 1.4, qL, qR)
    perm = [0, 2, 3, 1, 4, 5]                     # (u,v,w) -> (w,u,v): x-normal becomes y-normal
    qLy, qRy = qL[[0, 3, 1, 2, 4, 5]], qR[[0, 3, 1, 2, 4, 5]]
    Fy = O.hllc(1, 1.4, qLy, qRy)
    assert Fy[[0, 2, 3, 1, 4, 5]] == pytest.approx(Fx, rel=1e-15)
    assert perm


# ---------------------------------------------------------------- O8 dt (P11)
def test_dt_closed_form_uniform():
    gam = 5.0 / 3.0
    wl = W.uniform((8, 4, 16), (4, 4, 8), 0, (2.0, 0.3, -0.7, 0.1, 1.5), gamma=gam, cfl=0.4,
                   prob_hi=(1.0, 0.25, 4.0))
    U = W.initial_state(wl)
    dt = O.estimate_dt(O.make_params(wl.params), U)
    c = np.sqrt(gam * 1.5 / 2.0)
    ref = 0.4 / ((0.3 + c) * 8 + (0.7 + c) * 16 + (0.1 + c) * 4)
    assert dt == pytest.approx(ref, rel=1e-14)


def test_dt_takes_the_maximum_zone_and_flags_bad_state():
    wl = W.uniform((8, 8, 8), (4, 4, 4), 0, (1.0, 0.0, 0.0, 0.0, 1.0))
    U = W.initial_state(wl)
    p = O.make_params(wl.params)
    dt0 = O.estimate_dt(p, U)
    U5 = U.reshape(wl.state_shape)
    U5[5, W.EINT, 5, 6, 7] *= 4.0                 # one hot valid zone in the last-but-two box
    assert O.estimate_dt(p, U) == pytest.approx(dt0 / 2.0, rel=1e-14)
    U5[0, W.EINT, 0, 0, 0] = 1e30                 # ghost zones are not looked at
    assert O.estimate_dt(p, U) == pytest.approx(dt0 / 2.0, rel=1e-14)
    U5[3, W.MY, 5, 5, 5] = np.nan          # (a NaN density would be floored by max(), S8)
    rc, _ = O.estimate_dt_rc(p, U)
    assert rc == -4


# ---------------------------------------------------------------- O1 ghost fill (P12)
def _encode(c, gx, gy, gz):
    return c * 1.0e6 + gz * 1.0e4 + gy * 1.0e2 + gx + 1.0


@pytest.mark.parametrize("bcs", [(0, 0, 0), (1, 1, 1), (2, 2, 2), (1, 0, 2), (2, 1, 0)])
def test_ghost_fill_index_encoded(bcs):
    ndom, nbox, ng, ns = (8, 12, 8), (4, 6, 8), 4, 1
    wl = W.uniform(ndom, nbox, ns, (1, 0, 0, 0, 1), bc=bcs)
    nvar = wl.nvar
    G = np.empty((nvar, ndom[2], ndom[1], ndom[0]))
    gz, gy, gx = np.meshgrid(np.arange(ndom[2]), np.arange(ndom[1]), np.arange(ndom[0]), indexing="ij")
    for c in range(nvar):
        G[c] = _encode(c, gx, gy, gz)
    U = W.scatter_valid(wl, G, ghost_value=-777.0)
    O.fill_ghosts(O.make_params(wl.params), U)
    U = U.reshape(wl.state_shape)
    NB, nb = wl.NB, wl.nb

    def src(d, g):
        n = ndom[d]
        if 0 <= g < n: return g, 1
        if bcs[d] == 0: return g % n, 1
        if bcs[d] == 1: return min(max(g, 0), n - 1), 1
        return (-1 - g if g < 0 else 2 * n - 1 - g), -1

    for b in range(wl.nboxes):
        bi, bj, bk = b % NB[0], (b // NB[0]) % NB[1], b // (NB[0] * NB[1])
        for kl in range(wl.nt[2]):
            for jl in range(wl.nt[1]):
                for il in range(wl.nt[0]):
                    sx, fx = src(0, bi * nb[0] + il - ng)
                    sy, fy = src(1, bj * nb[1] + jl - ng)
                    sz, fz = src(2, bk * nb[2] + kl - ng)
                    for c in range(nvar):
                        ref = _encode(c, sx, sy, sz)
                        if c == 1: ref *= fx
                        if c == 2: ref *= fy
                        if c == 3: ref *= fz
                        assert U[b, c, kl, jl, il] == ref, (b, c, kl, jl, il)


def test_ghost_fill_rejects_bad_params():
    wl = W.uniform((8, 8, 8), (3, 4, 4), 0, (1, 0, 0, 0, 1))
    assert O.state_doubles(O.make_params(wl.params)) == 0          # nbox does not divide ndom
    wl = W.uniform((8, 8, 8), (4, 4, 4), 0, (1, 0, 0, 0, 1))
    wl.params["bc_lo"] = [0, 1, 1]; wl.params["bc_hi"] = [1, 1, 1]    # periodic on one side only
    assert O.state_doubles(O.make_params(wl.params)) == 0


# ---------------------------------------------------------------- O9 totals
def test_totals_exact_on_integers():
    wl = W.uniform((8, 8, 8), (4, 4, 4), 2, (1, 0, 0, 0, 1), prob_hi=(8.0, 8.0, 8.0))
    rng = np.random.default_rng(3)
    G = rng.integers(-1000, 1000, size=(wl.nvar, 8, 8, 8)).astype(np.float64)
    U = W.scatter_valid(wl, G, ghost_value=1e30)                     # ghosts must not be summed
    tot = O.conserved_totals(O.make_params(wl.params), U)
    ref = [G[c].sum() for c in (0, 1, 2, 3, 4, 6, 7)]               # rho*e (5) has no total
    assert np.array_equal(tot, ref)


def test_totals_compensated_sum():
    wl = W.uniform((8, 8, 8), (4, 4, 4), 0, (1, 0, 0, 0, 1), prob_hi=(8.0, 8.0, 8.0))
    G = np.zeros((6, 8, 8, 8)); G[0] = 1e-3; G[0, 0, 0, 0] = 1e16; G[0, 7, 7, 7] = -1e16
    tot = O.conserved_totals(O.make_params(wl.params), W.scatter_valid(wl, G))
    assert tot[0] == pytest.approx(510 * 1e-3, rel=1e-12)           # naive summation loses this

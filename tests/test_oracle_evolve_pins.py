"""Closed-form pins of the evolved internal-energy update O11 (readings G1-G5;
SURVEY 8(f) NEXT-1): L_e = -div(F_rho e) - p_c div(u_face) in the regime where the dual-energy switch
selects the evolved value.  Nothing here comes from the CUDA path.

P14  Uniform rho and rho*e, velocity LINEAR in each coordinate, u_d = U_d - a_d x_d, everything
     hypersonic (U_d >> c, so every face is upwind: F = F_L, u_face = n_L).  PPM reproduces linear data
     exactly (pin P5), so at interior faces u_face is the exact face value, div(u_face) = -(a_x+a_y+a_z)
     and F_e = rho u_face e.  One stage gives, per zone,
         rho*e_1 = rho*e_0 (1 + gamma A dt),   A = a_x + a_y + a_z
     (-div F_e contributes A rho*e, -p_c div u contributes (gamma-1) A rho*e: adiabatic compression,
     d(rho e)/dt = gamma A rho e).  With one non-zero rate a the state after stage 0 is again uniform rho,
     rho*e and linear u with rate a1 = a (1 + 2 a dt)/(1 + a dt), so the Heun value is the closed form
         rho*e_new = 1/2 rho*e_0 + 1/2 rho*e_0 (1 + gamma a dt)(1 + gamma a1 dt).
     A flipped sign of p_c div u gives (2 - gamma) instead of gamma; p_c taken from U0 instead of the stage
     state changes the Heun value by ~4e-6 relative; a dropped direction or a wrong dxinv changes A.
P15  Uniform rho, u; a STEP in e = rho*e/rho.  PPM leaves a step flat on both sides (pin P5), div(u_face) = 0,
     so one stage moves rho*e by the upwinded flux only: for u > 0 the zone right of the step changes by
     -dt rho u (e_R - e_L)/dx and its left neighbour does not change; for u < 0 the roles swap (upwind side
     of F_e, reading G1)."""
import numpy as np
import pytest

from oracle import oracle_binding as O
from paper_2007_05218_b200 import workloads as W

GAMMA = 1.4


def make(ndom, prob_hi, rho, vel, rhoe):
    """Single outflow box; vel = (u,v,w) arrays of shape (nz,ny,nx); rho, rhoe scalars or arrays."""
    wl = W.uniform(ndom, ndom, 0, (1.0, 0.0, 0.0, 0.0, 1.0), bc=W.OUTFLOW, gamma=GAMMA, prob_hi=prob_hi)
    wl.params["evolve_eint"] = 1
    shape = (ndom[2], ndom[1], ndom[0])
    G = np.zeros((6,) + shape)
    G[W.RHO] = rho
    for d in range(3):
        G[1 + d] = G[W.RHO] * vel[d]
    G[W.EINT] = rhoe
    G[W.EDEN] = G[W.EINT] + 0.5 * G[W.RHO] * (vel[0] ** 2 + vel[1] ** 2 + vel[2] ** 2)
    return wl, G


def centres(n, L):
    return (np.arange(n) + 0.5) * (L / n)


def test_p14_compression_one_stage_three_directions():
    # dyadic numbers: every face value, flux and difference below is exact in binary64
    ndom, L = (16, 16, 16), (0.25, 0.5, 1.0)                       # dx = 1/64, 1/32, 1/16: three different dxinv
    x, y, z = centres(16, L[0]), centres(16, L[1]), centres(16, L[2])
    a = (0.5, 0.25, -0.125)                                         # compression in x, y; expansion in z
    shape = (16, 16, 16)
    u = np.broadcast_to((1024.0 - a[0] * x)[None, None, :], shape)
    v = np.broadcast_to((2048.0 - a[1] * y)[None, :, None], shape)
    w = np.broadcast_to((512.0 - a[2] * z)[:, None, None], shape)
    rhoe0 = 2.0 ** -10
    wl, G = make(ndom, L, 1.0, (u, v, w), rhoe0)
    assert G[W.EINT].max() < 1e-8 * G[W.EDEN].min()                 # switch on everywhere (threshold 1e-4)
    U0 = W.scatter_valid(wl, G)
    U1 = np.zeros_like(U0)
    p = O.make_params(wl.params)
    dt = 2.0 ** -7
    O.fill_ghosts(p, U0)
    O.advance_stage(p, 0, dt, U0, U1)
    out = W.gather_valid(wl, U1)
    A = sum(a)
    inner = (slice(3, -3),) * 3                                     # outflow ghosts break linearity within 3 zones
    expect = rhoe0 * (1.0 + GAMMA * A * dt)
    assert np.abs(out[W.EINT][inner] - expect).max() <= 4e-16 * expect
    # the synchronised value rho*E - K would be useless here (K ~ 2.7e6, rounding of rho*E ~ 5e-10 >> rho*e ulp)
    assert np.abs(out[W.RHO][inner] - (1.0 + A * dt)).max() <= 1e-15


def test_p14_compression_heun_closed_form_each_direction():
    for d in range(3):
        ndom = [8, 8, 8]
        ndom[d] = 32
        L = [n / 64.0 for n in ndom]
        xc = centres(32, L[d])
        a, U, dt, rhoe0 = 0.5, 1024.0, 2.0 ** -7, 2.0 ** -10
        shape = (ndom[2], ndom[1], ndom[0])
        line = U - a * xc
        bshape = [1, 1, 1]
        bshape[2 - d] = 32
        vel = [np.zeros(shape), np.zeros(shape), np.zeros(shape)]
        vel[d] = np.broadcast_to(line.reshape(bshape), shape)
        wl, G = make(tuple(ndom), tuple(L), 1.0, vel, rhoe0)
        U0 = W.scatter_valid(wl, G)
        U1 = np.zeros_like(U0)
        O.step_fixed_dt(O.make_params(wl.params), U0, U1, dt)
        out = W.gather_valid(wl, U0)
        a1 = a * (1.0 + 2.0 * a * dt) / (1.0 + a * dt)
        expect = 0.5 * rhoe0 + 0.5 * rhoe0 * (1.0 + GAMMA * a * dt) * (1.0 + GAMMA * a1 * dt)
        sl = [slice(None)] * 3
        sl[2 - d] = slice(7, -7)                                    # two stages: 3 + 3 zones of influence, +1
        got = out[W.EINT][tuple(sl)]
        # stage 1 divides (rho u)_1 by rho_1: u_1 ~ 1e3 carries 1e-13 of rounding, times dxinv = 64 in div u
        assert np.abs(got - expect).max() <= 1e-10 * expect, d
        # the alternatives a plausible mistake would produce are far outside that tolerance
        wrong_sign = 0.5 * rhoe0 + 0.5 * rhoe0 * (1.0 + (2.0 - GAMMA) * a * dt) * (1.0 + (2.0 - GAMMA) * a1 * dt)
        base_pc = 0.5 * rhoe0 + 0.5 * (rhoe0 * (1.0 + GAMMA * a * dt) * (1.0 + a1 * dt) + dt * (GAMMA - 1.0) * rhoe0 * a1)
        assert abs(wrong_sign - expect) > 1e-4 * expect and abs(base_pc - expect) > 1e-7 * expect


@pytest.mark.parametrize("sign", [+1.0, -1.0])
def test_p15_step_in_e_is_upwinded_with_the_mass_flux(sign):
    ndom, L = (32, 4, 4), (0.5, 0.0625, 0.0625)                    # dx = 1/64
    shape = (4, 4, 32)
    u = np.full(shape, sign * 1024.0)
    zero = np.zeros(shape)
    rhoe = np.where(np.arange(32) < 16, 2.0 ** -10, 3.0 * 2.0 ** -10)[None, None, :] + zero
    wl, G = make(ndom, L, 1.0, (u, zero, zero), rhoe)
    U0 = W.scatter_valid(wl, G)
    U1 = np.zeros_like(U0)
    p = O.make_params(wl.params)
    dt = 2.0 ** -18
    O.fill_ghosts(p, U0)
    O.advance_stage(p, 0, dt, U0, U1)
    out = W.gather_valid(wl, U1)[W.EINT][0, 0]
    jump = 2.0 * 2.0 ** -10                                         # e_R - e_L (rho = 1)
    expect = rhoe[0, 0].copy()
    if sign > 0:
        expect[16] -= dt * 1024.0 * jump * 64.0                     # left value flows into the zone right of the step
    else:
        expect[15] += dt * 1024.0 * jump * 64.0                     # right value flows into the zone left of it
    assert np.array_equal(out, expect)

"""Pins of the optional evolved internal energy O11 (second half):
what the arithmetic fixes.  Where rho*E - K is a healthy fraction of rho*E the dual-energy switch selects it
and the scheme is bit-identical to the base scheme; in a uniform flow the evolved equation has a zero
right-hand side exactly; and at Mach 10^6 the synchronised value is limited by the rounding of rho*E while
the evolved one is not.  Nothing here comes from the CUDA path."""
import copy

import numpy as np

from oracle import oracle_binding as O
from paper_2007_05218_b200 import workloads as W
from test_oracle_scheme import run_steps


def evolved(wl):
    w = copy.deepcopy(wl)
    w.params["evolve_eint"] = 1
    return w


def test_evolve_is_bitwise_the_base_scheme_where_the_switch_is_off():
    # config 3 (Mach ~0.3), Sod and a small Sedov blast: rho*e / rho*E >> 1e-4 everywhere
    for n, kw, steps in ((3, dict(ndom=(32, 16, 16), nbox=(16, 8, 8), nspec=2), 2), (1, {}, 10),
                         (2, dict(ndom=(32, 32, 32), nbox=(16, 16, 32)), 5)):
        wl = W.config(n, **kw)
        U0 = W.initial_state(wl)
        A, B = U0.copy(), U0.copy()
        run_steps(wl, A, steps)
        run_steps(evolved(wl), B, steps)
        assert np.array_equal(A, B), n


def hypersonic(u, p=0.1, X=(1.0,)):
    return W.uniform((16, 8, 8), (8, 8, 8), len(X), (1.0, u, -0.6 * u, 0.3 * u, p), bc=W.PERIODIC, X=X)


def test_evolve_free_stream_is_exact_when_the_switch_is_on():
    wl = evolved(hypersonic(300.0))
    U0 = W.initial_state(wl)
    G0 = W.gather_valid(wl, U0)
    assert G0[W.EINT].max() < 1e-4 * G0[W.EDEN].min()               # the evolved branch is the one in use
    A = U0.copy()
    run_steps(wl, A, 5)
    assert np.array_equal(W.gather_valid(wl, A), G0)                # every component, rho*e included, bitwise


def test_evolve_beats_the_rounding_of_the_total_energy():
    # Mach ~ 3e6: K = 7.25e11, rho*e = 0.3075; rho*E = K + rho*e is rounded to a multiple of ulp(K) = 1.2e-4, so
    # rho*E - K recovers rho*e only to ~2e-4 relative -- the defect the dual-energy switch exists for
    wl0 = hypersonic(1.0e6, p=0.123)                                  # rho*e = 0.3075, not a multiple of that ulp
    U0 = W.initial_state(wl0)
    G0 = W.gather_valid(wl0, U0)
    A, B = U0.copy(), U0.copy()
    run_steps(wl0, A, 2)
    run_steps(evolved(wl0), B, 2)
    e0 = G0[W.EINT, 0, 0, 0]
    sync_err = np.abs(W.gather_valid(wl0, A)[W.EINT] - e0).max() / e0
    evol_err = np.abs(W.gather_valid(wl0, B)[W.EINT] - e0).max() / e0
    assert evol_err == 0.0
    assert sync_err > 1e-6


def test_evolve_conserves_and_is_decomposition_invariant_when_active():
    # cold supersonic flow (Mach ~ 100-600) with density, velocity and pressure structure, flattening on too
    wl = evolved(W.config(3, ndom=(32, 32, 32), nbox=(32, 32, 32), nspec=1))
    wl.params["flatten"] = 1
    G0 = W.gather_valid(wl, W.initial_state(wl))
    rho = G0[W.RHO]
    vel = G0[1:4] / rho * 200.0 + np.array([300.0, -150.0, 80.0])[:, None, None, None]
    G0[1:4] = rho * vel
    G0[W.EINT] = 0.05 * (1.0 + 0.2 * np.sin(np.arange(32) * 2 * np.pi / 32))[None, None, :]
    G0[W.EDEN] = G0[W.EINT] + 0.5 * rho * (vel ** 2).sum(axis=0)
    assert (G0[W.EINT] / G0[W.EDEN]).max() < 1e-4
    out, tots = [], []
    for nbox in [(32, 32, 32), (16, 16, 16), (8, 16, 32)]:
        w = W.with_boxes(wl, nbox)
        U = W.scatter_valid(w, G0)
        p = O.make_params(w.params)
        t0 = O.conserved_totals(p, U)
        run_steps(w, U, 3)
        t1 = O.conserved_totals(p, U)
        out.append(W.gather_valid(w, U))
        tots.append((t0, t1))
    assert np.array_equal(out[0], out[1]) and np.array_equal(out[0], out[2])
    t0, t1 = tots[0]
    scale = np.abs(W.gather_valid(wl, W.scatter_valid(wl, G0))[[0, 1, 2, 3, 4, 6]]).sum(axis=(1, 2, 3)) / 32 ** 3
    assert np.all(np.abs(t1 - t0) <= 1e-13 * scale)                 # rho, momenta, rho*E, rho*X: untouched by O11
    e = out[0][W.EINT]
    assert e.min() > 0.0 and np.isfinite(e).all()
    # and the evolved branch did act: the result differs from the synchronised scheme
    w0 = copy.deepcopy(wl); w0.params["evolve_eint"] = 0
    U = W.scatter_valid(w0, G0)
    run_steps(w0, U, 3)
    assert not np.array_equal(W.gather_valid(w0, U)[W.EINT], e)


def test_hllc_face_velocity():
    # G2: contact speed inside the fan (Sod interface: SM = 0.6761234037828133, pin P6), the upwind normal
    # velocity when the whole fan is on one side
    import ctypes as C
    L = O.lib()
    dp = C.POINTER(C.c_double)
    L.oracle_hllc_u.restype = None
    L.oracle_hllc_u.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, dp, dp, dp, dp]
    def uface(d, qL, qR):
        qL, qR = np.array(qL, float), np.array(qR, float)
        F, u = np.zeros(5), C.c_double()
        L.oracle_hllc_u(d, 1.4, 1e-12, 1e-14, 0, qL.ctypes.data_as(dp), qR.ctypes.data_as(dp), F.ctypes.data_as(dp), C.byref(u))
        return u.value
    assert abs(uface(0, [1, 0, 0, 0, 1], [0.125, 0, 0, 0, 0.1]) - 0.6761234037828133) < 1e-14
    assert uface(1, [1, 0.3, 5.0, 0.2, 1], [0.9, 0.1, 6.0, 0.0, 0.8]) == 5.0       # supersonic to the right: left state
    assert uface(2, [1, 0.3, 0.1, -5.0, 1], [0.9, 0.1, 0.0, -6.0, 0.8]) == -6.0    # supersonic to the left: right state
    assert uface(0, [1, 0.0, 0, 0, 1], [1, 0.0, 0, 0, 1]) == 0.0                   # symmetric states at rest

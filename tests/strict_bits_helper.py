"""Run by tests/test_gpu_strict.py in a subprocess with HYDRO_LIB pointing at the strict build
(-fmad=false -DHYDRO_STRICT): three RK2 steps through the five separate C-ABI calls must reproduce the
oracle BIT FOR BIT (every operation rounded separately, IEEE division and square root: the scheme's
definition, DESIGN.md sec. 2 "the two builds")."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import numpy as np  # noqa: E402

from oracle import oracle_binding as O  # noqa: E402
from paper_2007_05218_b200 import workloads as W  # noqa: E402
from paper_2007_05218_b200.binding import Hydro  # noqa: E402

CASES = [("cfg5_small", lambda: W.config(5, ndom=(64, 64, 64), nbox=(32, 32, 32))),
         ("cfg1_sod", lambda: W.config(1)),
         ("cfg4_small", lambda: W.config(4, ndom=(32, 32, 64), nbox=(16, 32, 32))),
         ("cfg2_small", lambda: W.config(2, ndom=(48, 48, 48), nbox=(24, 24, 48))),
         ("cfg3_odd_box", lambda: W.config(3, ndom=(54, 30, 14), nbox=(27, 15, 7), nspec=1))]
bad = []
for name, make in CASES:
    for opts in ({}, {"flatten": 1}, {"flatten": 1, "evolve_eint": 1}):
        wl = make()
        wl.params.update(opts)
        h = Hydro(wl.params)
        assert h.hydro_query(6) == (0 if name == "cfg3_odd_box" else 1), name   # chunk-lane x sweep where the rows allow
        U0 = W.initial_state(wl)
        h.upload(U0, 0)
        p = O.make_params(wl.params)
        Uo, T = U0.copy(), np.zeros_like(U0)
        dts_o = [O.step(p, Uo, T) for _ in range(3)]
        dts_g = [h.step_explicit() for _ in range(3)]
        G, Go = W.gather_valid(wl, h.download(0).reshape(U0.shape)), W.gather_valid(wl, Uo)
        ok = dts_o == dts_g and np.array_equal(G, Go)
        print(name, opts, "bitwise" if ok else "DIFFERS", flush=True)
        if not ok:
            bad.append((name, opts))
# the optional marching x kernels (HYDRO_XMARCH=1) are the same definition: bitwise too
os.environ["HYDRO_XMARCH"] = "1"
for name, make in CASES[:3]:
    wl = make()
    h = Hydro(wl.params)
    assert h.hydro_query(4) == 1, name
    U0 = W.initial_state(wl)
    h.upload(U0, 0)
    p = O.make_params(wl.params)
    Uo, T = U0.copy(), np.zeros_like(U0)
    dts_o = [O.step(p, Uo, T) for _ in range(3)]
    dts_g = h.hydro_step(3, all_dts=True)
    ok = dts_o == dts_g and np.array_equal(W.gather_valid(wl, h.download(0).reshape(U0.shape)), W.gather_valid(wl, Uo))
    print(name, "xmarch", "bitwise" if ok else "DIFFERS", flush=True)
    if not ok:
        bad.append((name, "xmarch"))
os.environ["HYDRO_XMARCH"] = "0"
# the one-zone-per-lane x sweep (k_sweep_x, HYDRO_XCHUNK=0; the default on these geometries is the chunk-lane
# kernel of sweep_xc.cuh, exercised by the first loop): bitwise too, with and without the options
os.environ["HYDRO_XCHUNK"] = "0"
for name, make in CASES[:3]:
    for opts in ({}, {"flatten": 1, "evolve_eint": 1}):
        wl = make()
        wl.params.update(opts)
        h = Hydro(wl.params)
        assert h.hydro_query(6) == 0, name
        U0 = W.initial_state(wl)
        h.upload(U0, 0)
        p = O.make_params(wl.params)
        Uo, T = U0.copy(), np.zeros_like(U0)
        dts_o = [O.step(p, Uo, T) for _ in range(3)]
        dts_g = h.hydro_step(3, all_dts=True)
        ok = dts_o == dts_g and np.array_equal(W.gather_valid(wl, h.download(0).reshape(U0.shape)), W.gather_valid(wl, Uo))
        print(name, opts, "k_sweep_x", "bitwise" if ok else "DIFFERS", flush=True)
        if not ok:
            bad.append((name, "k_sweep_x"))
os.environ["HYDRO_XCHUNK"] = "1"
# the CTU update O12: strict build == oracle_ctu_step, bit for bit
for name, make in CASES:
    wl = make()
    h = Hydro(wl.params)
    U0 = W.initial_state(wl)
    h.upload(U0, 0)
    p = O.make_params(wl.params)
    Uo, T = U0.copy(), np.zeros_like(U0)
    dts_o = [O.ctu_step(p, Uo, T) for _ in range(3)]
    dts_g = h.hydro_ctu_step(3, all_dts=True)
    ok = dts_o == dts_g and np.array_equal(W.gather_valid(wl, h.download(0).reshape(U0.shape)), W.gather_valid(wl, Uo))
    print(name, "ctu", "bitwise" if ok else "DIFFERS", flush=True)
    if not ok:
        bad.append((name, "ctu"))
sys.exit(1 if bad else 0)

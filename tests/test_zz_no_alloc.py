"""hydro_conserved_totals_static: the conservation totals for callers that are not allowed to allocate.

A simulation code of the kind the paper describes takes all its device memory from a pool it grabbed at start-up
(cudaMalloc inside the timestep loop is "disastrous").  A diagnostics routine, an in-situ monitor or a
plug-in called from inside such a code is lent a device pointer to the state and nothing more: it cannot reach the
host code's pool, its own cudaMalloc may fail because the pool already holds the device's memory, and it cannot
create a hydro handle (hydro_init needs a scratch buffer and pins host memory).  For those callers the library keeps
the reduction's partial sums in an array compiled into it (592 KiB per GPU, at most 27 species) and offers one call
that takes the state, an output array and a stream.

This file is named so that pytest collects it last: with `-x` a failure here cannot hide any other test.  The GPU
test makes no assumption about what ran before it (it passes alone in a fresh process and at the end of the suite):
the built-in array is shared by every call in the process and may hold anything when the test starts.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2007_05218_b200 import binding as B
from paper_2007_05218_b200 import build as build_mod
from paper_2007_05218_b200 import workloads as W

# two states of different shape, component count and block count, so that the second call finds the first call's
# partial sums in the shared array (1024 blocks x 18 components, then 105 blocks x 6 components, then the first again)
SHAPES = [
    lambda: W.config(5, ndom=(64, 64, 64), nbox=(32, 32, 32)),
    lambda: W.config(3, ndom=(54, 30, 14), nbox=(27, 15, 7), nspec=1),
]


@pytest.mark.gpu
def test_static_totals_equal_the_handle_path_on_calls_in_a_row():
    """Call after call on states of different shapes, each result checked against hydro_conserved_totals (the
    existing path, caller-provided scratch) on the same device data, to the 1e-13 of the other totals tests (S22),
    and against the oracle's sums of the same state."""
    import torch
    from oracle import oracle_binding as O

    build_mod.build()
    cases = []
    for make in SHAPES:
        wl = make()
        U0 = W.initial_state(wl, ghost_value=1e30)      # a sum that strays into a ghost zone is off by 1e30
        h = B.Hydro(wl.params)
        h.upload(U0, 0)
        G = W.gather_valid(wl, np.abs(U0))
        scale = np.array([G[c if c < 5 else c + 1].sum() for c in range(wl.nflux)]) * np.prod(wl.dx)
        cases.append((wl, U0, h, scale))
    for wl, U0, h, scale in (cases[0], cases[1], cases[0]):
        want = np.array(h.hydro_conserved_totals(0))
        out = torch.full((wl.nflux,), float("nan"), dtype=torch.float64, device=h.U0.device)
        B.hydro_conserved_totals_static(h.p, h.U0, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert np.all(np.isfinite(got)), got
        assert np.all(np.abs(got - want) <= 1e-13 * scale), (got, want)
        ref = O.conserved_totals(O.make_params(wl.params), U0)
        assert np.all(np.abs(got - ref) <= 1e-13 * scale), (got, ref)


def test_static_totals_refuse_more_species_than_the_builtin_array_holds():
    """28 species = 33 conserved components, one more than the built-in array has room for: HYDRO_ENOMEM and a
    message that names the limit, decided before any CUDA call (so this runs without a GPU); 27 species pass that
    check and fail later, on the null pointers."""
    build_mod.build()
    L = B.lib()
    wl = W.config(3, ndom=(16, 16, 16), nbox=(8, 8, 8), nspec=28)
    rc = L.hydro_conserved_totals_static(C.byref(B.make_params(wl.params)), 256, 512, None)
    msg = L.hydro_last_error(None).decode()
    assert rc == B.HYDRO_ENOMEM, (rc, msg)
    assert "27" in msg and "hydro_conserved_totals " in msg, msg
    wl = W.config(3, ndom=(16, 16, 16), nbox=(8, 8, 8), nspec=27)
    rc = L.hydro_conserved_totals_static(C.byref(B.make_params(wl.params)), None, None, None)
    assert rc == B.HYDRO_EINVAL, (rc, L.hydro_last_error(None).decode())

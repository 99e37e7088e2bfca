"""The optional marching x kernels (march_x.cuh, HYDRO_XMARCH=1 at hydro_init; include/hydro.h lists the
switch) against the oracle: the same tolerances as the default lane-parallel x sweep, on geometries that
take them (nbox[0] % 4 == 0, even ng >= 4, 128 % nbox[1] == 0 or nbox[1] % 128 == 0) -- several row
tiles per k plane, a k extent that does not fill the last row tile, the shortest row, wide ghosts."""
import numpy as np
import pytest

from oracle import oracle_binding as O
from paper_2007_05218_b200 import workloads as W
from parity_util import rel_err
from test_gpu_parity import CASES

pytestmark = pytest.mark.gpu

XCASES = ["cfg1_sod", "cfg4_atmosphere_small", "cfg5_scaling_small", "cfg2_sedov_wide_rows", "cfg5_256_wide_box",
          "cfg2_ng6_no_species", "cfg5_tall_box", "cfg3_xmarch_ragged_k"]


@pytest.fixture
def xmarch(monkeypatch):
    monkeypatch.setenv("HYDRO_XMARCH", "1")      # read once per hydro_init


@pytest.mark.parametrize("name", XCASES)
def test_xmarch_one_step_and_five_steps(name, xmarch):
    from paper_2007_05218_b200.binding import Hydro
    wl = CASES[name]()
    U0 = W.initial_state(wl, ghost_value=np.nan)
    p = O.make_params(wl.params)
    h = Hydro(wl.params)
    assert h.hydro_query(4) == 1, "geometry was expected to take the marching x kernels"
    h.upload(U0, 0)
    Uo, T = U0.copy(), np.zeros_like(U0)
    dt_o = O.step(p, Uo, T)
    dt_g = h.step_explicit()
    assert abs(dt_g - dt_o) <= 1e-14 * dt_o
    e = rel_err(wl, h.download(0).reshape(U0.shape), Uo)
    assert np.all(e <= 1e-12), e
    dts_o = [O.step(p, Uo, T) for _ in range(4)]
    dts_g = h.hydro_step(4, all_dts=True)
    assert all(abs(a - b) <= 1e-12 * b for a, b in zip(dts_g, dts_o))
    e = rel_err(wl, h.download(0).reshape(U0.shape), Uo)
    assert np.all(e <= 1e-10), e


def test_default_is_the_lane_parallel_sweep():
    from paper_2007_05218_b200.binding import Hydro
    assert Hydro(CASES["cfg5_scaling_small"]().params).hydro_query(4) == 0

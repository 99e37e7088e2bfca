"""The chunk-lane x sweep (sweep_xc.cuh: a lane owns a 4-zone chunk of the flattened valid rows of a box; the
default where ng and nbox[0] are multiples of 4) against the oracle and against the one-zone-per-lane
k_sweep_x (HYDRO_XCHUNK=0; include/hydro.h lists the switch): rows shorter than a warp's 30 chunks (several
rows per warp), a chunk sequence that does not fill the last warp, ng = 8, no species / one / 13, both options."""
import numpy as np
import pytest

from oracle import oracle_binding as O
from paper_2007_05218_b200 import workloads as W
from parity_util import rel_err
from test_gpu_parity import CASES, with_ng

pytestmark = pytest.mark.gpu

XCASES = {
    "cfg1_sod": (CASES["cfg1_sod"], {}),
    "cfg4_atmosphere_small": (CASES["cfg4_atmosphere_small"], {}),
    "cfg5_scaling_small": (CASES["cfg5_scaling_small"], {}),
    "cfg5_256_wide_box": (CASES["cfg5_256_wide_box"], {}),
    "cfg5_tall_box": (CASES["cfg5_tall_box"], {}),
    "cfg3_short_rows": (lambda: W.config(3, ndom=(8, 20, 12), nbox=(4, 10, 6)), {}),
    "cfg2_ng8_no_species": (lambda: with_ng(W.config(2, ndom=(32, 32, 32), nbox=(32, 16, 16)), 8), {}),
    "cfg3_flatten": (lambda: W.config(3, ndom=(40, 32, 24), nbox=(20, 16, 12), nspec=3), {"flatten": 1}),
    "cfg2_flatten_evolve": (CASES["cfg2_sedov_small"], {"flatten": 1, "evolve_eint": 1}),
    "cfg4_evolve": (CASES["cfg4_atmosphere_small"], {"evolve_eint": 1}),
}


def run(wl, U0, nsteps):
    from paper_2007_05218_b200.binding import Hydro
    h = Hydro(wl.params)
    h.upload(U0, 0)
    dts = [h.step_explicit()]
    if nsteps > 1:
        dts += h.hydro_step(nsteps - 1, all_dts=True)
    return h, dts, h.download(0).reshape(U0.shape)


@pytest.mark.parametrize("name", list(XCASES))
def test_chunk_lane_x_sweep(name, monkeypatch):
    make, opts = XCASES[name]
    wl = make()
    wl.params.update(opts)
    U0 = W.initial_state(wl, ghost_value=np.nan)
    h, dts_c, Uc = run(wl, U0, 4)
    assert h.hydro_query(6) == 1, "geometry was expected to take the chunk-lane x sweep"
    p = O.make_params(wl.params)
    Uo, T = U0.copy(), np.zeros_like(U0)
    dts_o = [O.step(p, Uo, T) for _ in range(4)]
    assert all(abs(a - b) <= 1e-12 * b for a, b in zip(dts_c, dts_o))
    e = rel_err(wl, Uc, Uo)
    assert np.all(e <= (1e-10 if opts else 1e-11)), e
    # the same four steps with k_sweep_x: the same arithmetic on the same operands (FMA contraction may differ
    # between the two kernels in the default build, hence not bitwise here; bitwise in the strict build)
    monkeypatch.setenv("HYDRO_XCHUNK", "0")
    h0, dts_0, U0x = run(wl, U0, 4)
    assert h0.hydro_query(6) == 0
    assert all(abs(a - b) <= 1e-13 * b for a, b in zip(dts_c, dts_0))
    assert np.all(rel_err(wl, Uc, U0x) <= (1e-10 if opts else 1e-12))


def test_rows_that_are_not_whole_chunks_keep_the_lane_parallel_sweep():
    from paper_2007_05218_b200.binding import Hydro
    assert Hydro(CASES["cfg3_one_species_odd_box"]().params).hydro_query(6) == 0
    assert Hydro(CASES["cfg2_ng6_no_species"]().params).hydro_query(6) == 0
    assert Hydro(CASES["cfg3_ragged_rows"]().params).hydro_query(6) == 1

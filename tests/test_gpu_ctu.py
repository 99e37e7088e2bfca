"""GPU parity of the CTU update O12 (hydro_ctu_step, csrc/ctu.cuh) against oracle_ctu_step on the same seeded
inputs: <= 1e-12 after one step, <= 1e-10 after ten, dt to 1e-14 / 1e-12 (the north_star tolerances of the
method-of-lines path), free stream and the batching of boxes bitwise."""
import numpy as np
import pytest

from oracle import oracle_binding as O
from paper_2007_05218_b200 import workloads as W
from parity_util import rel_err
from test_gpu_parity import CASES

pytestmark = pytest.mark.gpu

CTU_CASES = [("cfg1_sod", 20), ("cfg2_sedov_small", 10), ("cfg3_periodic_small", 10), ("cfg4_atmosphere_small", 10),
             ("cfg5_scaling_small", 5), ("cfg3_one_species_odd_box", 3), ("cfg3_ng3", 3), ("cfg2_ng6_no_species", 3),
             ("cfg5_256_wide_box", 3)]


def hydro(wl):
    from paper_2007_05218_b200.binding import Hydro
    return Hydro(wl.params)


@pytest.mark.parametrize("name,nsteps", CTU_CASES)
def test_ctu_one_step_and_many(name, nsteps):
    wl = CASES[name]()
    U0 = W.initial_state(wl, ghost_value=np.nan)
    p = O.make_params(wl.params)
    h = hydro(wl)
    h.upload(U0, 0)
    Uo, T = U0.copy(), np.zeros_like(U0)
    dt_o = O.ctu_step(p, Uo, T)
    dt_g = h.hydro_ctu_step(1)                                  # odd number of steps: result copied back into U0
    assert abs(dt_g - dt_o) <= 1e-14 * dt_o
    e = rel_err(wl, h.download(0).reshape(U0.shape), Uo)
    assert np.all(e <= 1e-12), e
    dts_o = [O.ctu_step(p, Uo, T) for _ in range(nsteps - 1)]
    dts_g = h.hydro_ctu_step(nsteps - 1, all_dts=True)
    assert all(abs(a - b) <= 1e-12 * b for a, b in zip(dts_g, dts_o))
    e = rel_err(wl, h.download(0).reshape(U0.shape), Uo)
    assert np.all(e <= 1e-10), e


def test_ctu_batches_of_boxes_are_bitwise_the_same():
    import torch
    wl = CASES["cfg5_scaling_small"]()                          # 8 boxes
    U0 = W.initial_state(wl)
    hs = [hydro(wl) for _ in range(3)]
    for h, nb in zip(hs, (1, 3, 8)):                            # one box at a time, ragged batches, all at once
        h.upload(U0, 0)
        h.hydro_ctu_step(4, batch_boxes=nb)
    assert torch.equal(hs[0].U0, hs[1].U0) and torch.equal(hs[0].U0, hs[2].U0)


def test_ctu_free_stream_bitwise_and_conservation():
    wl = W.uniform((16, 16, 24), (8, 16, 12), 2, (1.3, 0.7, -0.4, 0.25, 0.9), bc=(W.OUTFLOW, W.PERIODIC, W.OUTFLOW), X=(0.3, 0.7))
    U0 = W.initial_state(wl, ghost_value=np.nan)
    h = hydro(wl)
    h.upload(U0, 0)
    h.hydro_ctu_step(3)
    G, G0 = W.gather_valid(wl, h.download(0).reshape(U0.shape)), W.gather_valid(wl, U0)
    keep = [c for c in range(wl.nvar) if c != W.EINT]
    assert np.array_equal(G[keep], G0[keep])
    wl = CASES["cfg3_periodic_small"]()
    U0 = W.initial_state(wl)
    h = hydro(wl)
    h.upload(U0, 0)
    t0 = np.array(h.hydro_conserved_totals(0))
    h.hydro_ctu_step(10)
    t1 = np.array(h.hydro_conserved_totals(0))
    absU = W.gather_valid(wl, np.abs(U0))
    scale = np.array([absU[c if c < 5 else c + 1].sum() * np.prod(wl.dx) for c in range(wl.nflux)])
    assert np.all(np.abs(t1 - t0) <= 1e-13 * scale)


def test_ctu_refuses_what_it_does_not_cover():
    from paper_2007_05218_b200 import binding as B
    wl = CASES["cfg5_scaling_small"]()
    wl.params["flatten"] = 1
    h = hydro(wl)
    with pytest.raises(B.HydroError) as ei:
        h.hydro_ctu_step(1)
    assert ei.value.code == B.HYDRO_EINVAL
    wl = CASES["cfg5_scaling_small"]()
    h = hydro(wl)
    import ctypes as C
    import torch
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    assert B.lib().hydro_ctu_step(h.h, small.data_ptr(), 1024, 1, None) == B.HYDRO_ENOMEM
    assert B.lib().hydro_ctu_step(h.h, None, 0, 1, None) == B.HYDRO_EINVAL
    assert B.hydro_ctu_scratch_bytes(B.make_params(wl.params)) == 12 * 18 * 40 ** 3 * 8

"""Two levels of refinement (second half): a coarse level and ONE
rectangular patch refined by 2 or 4, each with its own handle of the C ABI.  Plumbing only: the order of the calls.

One RK2 step with a common dt (no subcycling, no refluxing):
    dt = min(estimate_dt(coarse), estimate_dt(fine))
    for stage in 0, 1:
        fill_ghosts(coarse); fill_ghosts(fine)             # fine-fine and physical ghosts of the patch
        fill_from_coarse(fine <- coarse)                   # the patch's outer ghosts, conservative linear interpolation
        advance_stage(coarse); advance_stage(fine)
    average_down(coarse <- fine)                           # the coarse zones under the patch follow the fine solution
"""
from __future__ import annotations

import copy

BC_EXTERNAL = 3


def patch_params(coarse_params: dict, lo, extent, ratio: int, nbox) -> dict:
    """hydro_params of the patch covering coarse zones [lo, lo + extent) refined by `ratio`, in boxes of `nbox` fine zones."""
    p = copy.deepcopy(coarse_params)
    p["dx"] = [0.0, 0.0, 0.0]
    for d in range(3):
        dx = coarse_params.get("dx", (0.0, 0.0, 0.0))[d] or \
            (coarse_params["prob_hi"][d] - coarse_params["prob_lo"][d]) / coarse_params["ndom"][d]
        p["dx"][d] = dx / ratio          # exactly the coarse zone width over 2 or 4, whatever the patch's own extent gives
        if lo[d] < 0 or lo[d] + extent[d] > coarse_params["ndom"][d]:
            raise ValueError("the patch must lie inside the coarse domain")
        p["ndom"][d] = ratio * extent[d]
        p["nbox"][d] = nbox[d]
        p["prob_lo"][d] = coarse_params["prob_lo"][d] + lo[d] * dx
        p["prob_hi"][d] = coarse_params["prob_lo"][d] + (lo[d] + extent[d]) * dx
        on_lo = lo[d] == 0 and coarse_params["bc_lo"][d] != 0
        on_hi = lo[d] + extent[d] == coarse_params["ndom"][d] and coarse_params["bc_hi"][d] != 0
        p["bc_lo"][d] = coarse_params["bc_lo"][d] if on_lo else BC_EXTERNAL
        p["bc_hi"][d] = coarse_params["bc_hi"][d] if on_hi else BC_EXTERNAL
    return p


class TwoLevelHydro:
    def __init__(self, coarse_params: dict, lo, extent, ratio: int, nbox_fine, device="cuda:0"):
        from .binding import Hydro
        self.lo, self.ratio = tuple(int(x) for x in lo), int(ratio)
        self.fine_params = patch_params(coarse_params, lo, extent, ratio, nbox_fine)
        self.coarse = Hydro(coarse_params, device=device)
        self.fine = Hydro(self.fine_params, device=device)

    def step(self) -> float:
        c, f = self.coarse, self.fine
        dt = min(c.hydro_estimate_dt(), f.hydro_estimate_dt())
        for stage in (0, 1):
            c.hydro_fill_ghosts(stage)
            f.hydro_fill_ghosts(stage)
            f.hydro_fill_from_coarse(stage, c, stage, self.lo, self.ratio)
            c.hydro_advance_stage(stage, dt)
            f.hydro_advance_stage(stage, dt)
        c.hydro_average_down(0, f, 0, self.lo, self.ratio)
        return dt

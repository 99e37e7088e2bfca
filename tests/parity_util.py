"""Comparison metric of SURVEY.md 8(c) S16 and small helpers shared by the GPU parity tests."""
import numpy as np

from paper_2007_05218_b200 import workloads as W


def rel_err(wl, Ug, Uo):
    """max over valid zones of |gpu - oracle| / scale_c per stored component; the three momenta
    share one scale max(|rho u|,|rho v|,|rho w|, |rho|*|c|); a component that is identically zero in
    the oracle must be exactly zero on the GPU (err = 0 or inf)."""
    Gg, Go = W.gather_valid(wl, Ug), W.gather_valid(wl, Uo)
    gam = wl.params["gamma"]
    rho = np.maximum(Go[W.RHO], 1e-300)
    cs = np.sqrt(gam * np.maximum((gam - 1.0) * Go[W.EINT], 0.0) / rho)
    mom_scale = max(np.abs(Go[W.MX]).max(), np.abs(Go[W.MY]).max(), np.abs(Go[W.MZ]).max(),
                    np.abs(Go[W.RHO]).max() * cs.max())
    errs = np.zeros(wl.nvar)
    for c in range(wl.nvar):
        scale = mom_scale if c in (W.MX, W.MY, W.MZ) else np.abs(Go[c]).max()
        diff = np.abs(Gg[c] - Go[c]).max()
        if not np.all(np.isfinite(Gg[c])):
            errs[c] = np.inf
        elif scale == 0.0:
            errs[c] = 0.0 if diff == 0.0 else np.inf
        else:
            errs[c] = diff / scale
    return errs


def oracle_run(O, wl, U0, nsteps):
    p = O.make_params(wl.params)
    U1 = np.zeros_like(U0)
    return [O.step(p, U0, U1) for _ in range(nsteps)]

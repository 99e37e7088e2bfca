"""Thin Python binding of libhydro_b200.so (include/hydro.h): argument marshalling only.

Same names as the C ABI.  PyTorch is used for device memory and the CUDA stream; every
step of the path runs in the library's kernels.  There is no CPU fallback: if the shared
library is missing this module raises at first use.
"""
from __future__ import annotations

import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("HYDRO_LIB") or os.path.join(HERE, "libhydro_b200.so")

HYDRO_OK, HYDRO_EINVAL, HYDRO_ENOMEM, HYDRO_ECUDA, HYDRO_ESTATE = 0, -1, -2, -3, -4
EXPORTS = ["hydro_state_bytes", "hydro_scratch_bytes", "hydro_init", "hydro_fill_ghosts",
           "hydro_advance_stage", "hydro_estimate_dt", "hydro_conserved_totals", "hydro_step",
           "hydro_launch_count", "hydro_query", "hydro_profile", "hydro_profile_read", "hydro_destroy", "hydro_last_error", "hydro_run_host",
           "hydro_halo_bytes", "hydro_pack_halo", "hydro_unpack_halo", "hydro_ctu_scratch_bytes", "hydro_ctu_step", "hydro_fill_from_coarse", "hydro_average_down",
           "hydro_conserved_totals_static"]
PROBE_LIB_PATH = os.path.join(HERE, "libhydro_probe_b200.so")
PROBE_EXPORTS = ["hydro_probe_fp64"]


class HydroParams(C.Structure):
    """Mirror of `hydro_params` in include/hydro.h."""
    _fields_ = [
        ("ndom", C.c_int32 * 3), ("nbox", C.c_int32 * 3), ("ng", C.c_int32), ("nspec", C.c_int32),
        ("bc_lo", C.c_int32 * 3), ("bc_hi", C.c_int32 * 3),
        ("prob_lo", C.c_double * 3), ("prob_hi", C.c_double * 3),
        ("gamma", C.c_double), ("cfl", C.c_double), ("grav", C.c_double * 3),
        ("small_dens", C.c_double), ("small_pres", C.c_double),
        ("flatten", C.c_int32), ("evolve_eint", C.c_int32),
        ("dx", C.c_double * 3),
    ]


def make_params(d: dict) -> HydroParams:
    p = HydroParams()
    for k in ("ndom", "nbox", "bc_lo", "bc_hi"):
        setattr(p, k, (C.c_int32 * 3)(*[int(x) for x in d[k]]))
    for k in ("prob_lo", "prob_hi", "grav"):
        setattr(p, k, (C.c_double * 3)(*[float(x) for x in d[k]]))
    p.ng, p.nspec = int(d["ng"]), int(d["nspec"])
    p.gamma, p.cfl = float(d["gamma"]), float(d["cfl"])
    p.small_dens, p.small_pres = float(d.get("small_dens", 1e-12)), float(d.get("small_pres", 1e-14))
    p.flatten = int(d.get("flatten", 0))
    p.evolve_eint = int(d.get("evolve_eint", 0))
    p.dx = (C.c_double * 3)(*[float(x) for x in d.get("dx", (0.0, 0.0, 0.0))])
    return p


class HydroError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"hydro error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libhydro_b200.so and declare every entry point of include/hydro.h."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2007_05218_b200.build` "
                          "(there is no CPU fallback for the hydro path)")
    L = C.CDLL(LIB_PATH)
    pp, vp, dp = C.POINTER(HydroParams), C.c_void_p, C.POINTER(C.c_double)
    L.hydro_state_bytes.restype = C.c_size_t
    L.hydro_state_bytes.argtypes = [pp]
    L.hydro_scratch_bytes.restype = C.c_size_t
    L.hydro_scratch_bytes.argtypes = [pp]
    L.hydro_init.argtypes = [pp, vp, vp, vp, C.c_size_t, vp, C.POINTER(vp)]
    L.hydro_fill_ghosts.argtypes = [vp, C.c_int]
    L.hydro_advance_stage.argtypes = [vp, C.c_int, C.c_double]
    L.hydro_estimate_dt.argtypes = [vp, dp]
    L.hydro_conserved_totals.argtypes = [vp, C.c_int, dp]
    L.hydro_step.argtypes = [vp, C.c_int, dp]
    L.hydro_query.argtypes = [vp, C.c_int]
    L.hydro_launch_count.restype = C.c_longlong
    L.hydro_launch_count.argtypes = [vp]
    L.hydro_profile.argtypes = [vp, C.c_int]
    L.hydro_profile_read.argtypes = [vp, dp, C.POINTER(C.c_longlong)]
    L.hydro_destroy.argtypes = [vp]
    L.hydro_last_error.restype = C.c_char_p
    L.hydro_last_error.argtypes = [vp]
    L.hydro_run_host.argtypes = [pp, vp, C.c_int, dp, dp]
    L.hydro_ctu_scratch_bytes.restype = C.c_size_t
    L.hydro_ctu_scratch_bytes.argtypes = [pp]
    L.hydro_ctu_step.argtypes = [vp, vp, C.c_size_t, C.c_int, dp]
    L.hydro_fill_from_coarse.argtypes = [vp, C.c_int, vp, C.c_int, C.POINTER(C.c_int32), C.c_int]
    L.hydro_average_down.argtypes = [vp, C.c_int, vp, C.c_int, C.POINTER(C.c_int32), C.c_int]
    L.hydro_halo_bytes.restype = C.c_size_t
    L.hydro_halo_bytes.argtypes = [pp, C.c_int]
    L.hydro_pack_halo.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp]
    L.hydro_unpack_halo.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp]
    L.hydro_conserved_totals_static.argtypes = [pp, vp, vp, vp]
    _lib = L
    return L


def hydro_state_bytes(p: HydroParams) -> int:
    return lib().hydro_state_bytes(C.byref(p))


def hydro_scratch_bytes(p: HydroParams) -> int:
    return lib().hydro_scratch_bytes(C.byref(p))


def hydro_ctu_scratch_bytes(p: HydroParams) -> int:
    return lib().hydro_ctu_scratch_bytes(C.byref(p))


def hydro_halo_bytes(p: HydroParams, dim: int) -> int:
    return lib().hydro_halo_bytes(C.byref(p), dim)


def hydro_conserved_totals_static(p: HydroParams, U_dev, totals_dev, stream=None):
    """Conserved totals of a device-resident state for code that must not allocate (include/hydro.h): no handle, no
    scratch buffer; the reduction's partial sums live in an array built into the library (nspec <= 27).

    U_dev: CUDA float64 tensor holding one state in layout a1; totals_dev: CUDA float64 tensor of 5 + nspec
    elements on the same device, written by the call; stream: a torch.cuda.Stream of that device (default: the
    device's current stream).  Asynchronous: synchronise the stream before reading totals_dev.  This wrapper
    allocates nothing on the device either; both tensors are the caller's."""
    import torch
    if stream is None:
        stream = torch.cuda.current_stream(U_dev.device)
    rc = lib().hydro_conserved_totals_static(C.byref(p), U_dev.data_ptr(), totals_dev.data_ptr(), stream.cuda_stream)
    if rc != 0:
        raise HydroError(rc, lib().hydro_last_error(None).decode())


_probe = None


def probe_lib():
    """Load libhydro_probe_b200.so (include/hydro_probe.h): bench.py's measurement aid, not the product."""
    global _probe
    if _probe is None:
        if not os.path.exists(PROBE_LIB_PATH):
            raise ImportError(f"{PROBE_LIB_PATH} is missing: run `python -m paper_2007_05218_b200.build`")
        _probe = C.CDLL(PROBE_LIB_PATH)
        _probe.hydro_probe_fp64.argtypes = [C.POINTER(C.c_double)]
    return _probe


def hydro_probe_fp64():
    """FP64 thread-instructions per second of the three probe kernels (include/hydro_probe.h)."""
    r = (C.c_double * 3)()
    rc = probe_lib().hydro_probe_fp64(r)
    if rc != 0:
        raise HydroError(rc, "hydro_probe_fp64 failed")
    return {"dfma": r[0], "dadd_dmul": r[1], "dfma_with_imad": r[2]}


def hydro_run_host(p: HydroParams, U_host, nsteps: int, want_totals: bool = False):
    """U_host: numpy float64 array or CPU torch tensor in layout a1, advanced in place.
    Returns (dts, totals-or-None)."""
    ptr = U_host.ctypes.data if hasattr(U_host, "ctypes") else U_host.data_ptr()
    dts = (C.c_double * max(nsteps, 1))()
    tot = (C.c_double * (5 + p.nspec))()
    rc = lib().hydro_run_host(C.byref(p), ptr, nsteps, dts, tot if want_totals else None)
    if rc != 0:
        raise HydroError(rc, lib().hydro_last_error(None).decode())
    return list(dts)[:nsteps], (list(tot) if want_totals else None)


class Hydro:
    """Owns the device buffers (torch) and a handle; methods are the C-ABI calls."""

    def __init__(self, params: dict | HydroParams, device="cuda:0", stream=None):
        import torch
        self.torch = torch
        self.p = params if isinstance(params, HydroParams) else make_params(params)
        L = lib()
        sb, scb = hydro_state_bytes(self.p), hydro_scratch_bytes(self.p)
        if sb == 0:
            raise HydroError(HYDRO_EINVAL, "invalid hydro_params")
        self.device = torch.device(device)
        self.nflux = 5 + self.p.nspec
        self.h = C.c_void_p()
        with torch.cuda.device(self.device):
            self.U0 = torch.empty(sb // 8, dtype=torch.float64, device=self.device)
            self.U1 = torch.zeros(sb // 8, dtype=torch.float64, device=self.device)
            self.scratch = torch.empty(scb, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            rc = L.hydro_init(C.byref(self.p), self.U0.data_ptr(), self.U1.data_ptr(), self.scratch.data_ptr(),
                              scb, self.stream.cuda_stream, C.byref(self.h))
        if rc != 0:
            raise HydroError(rc, L.hydro_last_error(None).decode())

    def _check(self, rc):
        if rc != 0:
            raise HydroError(rc, lib().hydro_last_error(self.h).decode())

    # ---- state transfer (plumbing) ----
    def upload(self, U_host, which=0):
        t = self.torch.as_tensor(U_host).reshape(-1)
        (self.U0 if which == 0 else self.U1).copy_(t, non_blocking=False)

    def download(self, which=0):
        return (self.U0 if which == 0 else self.U1).cpu().numpy()

    # ---- the C-ABI calls ----
    def hydro_fill_ghosts(self, which):
        self._check(lib().hydro_fill_ghosts(self.h, which))

    def hydro_advance_stage(self, stage, dt):
        self._check(lib().hydro_advance_stage(self.h, stage, dt))

    def hydro_estimate_dt(self):
        out = C.c_double(0.0)
        self._check(lib().hydro_estimate_dt(self.h, C.byref(out)))
        return out.value

    def hydro_conserved_totals(self, which=0):
        out = (C.c_double * self.nflux)()
        self._check(lib().hydro_conserved_totals(self.h, which, out))
        return list(out)

    def hydro_step(self, nsteps=1, want_dt=True, all_dts=False):
        """nsteps RK2 steps in one call.  Returns the last dt (want_dt), every dt (all_dts) or None."""
        out = (C.c_double * max(nsteps, 1))()
        self._check(lib().hydro_step(self.h, nsteps, out if (want_dt or all_dts) else None))
        if all_dts:
            return list(out)[:nsteps]
        return out[nsteps - 1] if (want_dt and nsteps > 0) else (0.0 if want_dt else None)

    def hydro_ctu_step(self, nsteps=1, batch_boxes=None, all_dts=False):
        """nsteps CTU steps (O12).  The scratch for `batch_boxes` boxes (default: as many as fit in 40 GB, at least
        one) is allocated on first use and kept."""
        per_box = lib().hydro_ctu_scratch_bytes(C.byref(self.p))
        nboxes = 1
        for d in range(3):
            nboxes *= self.p.ndom[d] // self.p.nbox[d]
        nb = batch_boxes or max(1, min(nboxes, int(40e9 // per_box)))
        if getattr(self, "_ctu", None) is None or self._ctu.numel() < nb * per_box:
            self._ctu = self.torch.empty(nb * per_box, dtype=self.torch.uint8, device=self.device)
        out = (C.c_double * max(nsteps, 1))()
        self._check(lib().hydro_ctu_step(self.h, self._ctu.data_ptr(), nb * per_box, nsteps, out))
        return list(out)[:nsteps] if all_dts else (out[nsteps - 1] if nsteps > 0 else 0.0)

    def hydro_fill_from_coarse(self, which, coarse, which_coarse, lo_coarse, ratio):
        """self = the refined patch; coarse = the Hydro of the coarse level (include/hydro.h, O13)."""
        lo = (C.c_int32 * 3)(*[int(x) for x in lo_coarse])
        self._check(lib().hydro_fill_from_coarse(self.h, which, coarse.h, which_coarse, lo, int(ratio)))

    def hydro_average_down(self, which, fine, which_fine, lo_coarse, ratio):
        """self = the coarse level; fine = the Hydro of the refined patch (include/hydro.h, O13 restriction)."""
        lo = (C.c_int32 * 3)(*[int(x) for x in lo_coarse])
        self._check(lib().hydro_average_down(self.h, which, fine.h, which_fine, lo, int(ratio)))

    def hydro_pack_halo(self, which, dim, side, buf):
        """buf: device tensor of hydro_halo_bytes(params, dim) bytes (sharded.py)."""
        self._check(lib().hydro_pack_halo(self.h, which, dim, side, buf.data_ptr()))

    def hydro_unpack_halo(self, which, dim, side, buf):
        self._check(lib().hydro_unpack_halo(self.h, which, dim, side, buf.data_ptr()))

    def hydro_launch_count(self):
        return lib().hydro_launch_count(self.h)

    def hydro_query(self, what):
        return lib().hydro_query(self.h, what)

    KERNEL_CLASSES = ["fill_ghosts", "estimate_dt", "sweep_x", "hydro_y", "species_y", "hydro_z", "species_z",
                      "totals", "flatten", "ctu"]

    def hydro_profile(self, enable):
        self._check(lib().hydro_profile(self.h, int(enable)))

    def hydro_profile_read(self):
        ms = (C.c_double * 10)()
        cnt = (C.c_longlong * 10)()
        self._check(lib().hydro_profile_read(self.h, ms, cnt))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(self.KERNEL_CLASSES)}

    def step_explicit(self):
        """One RK2 step through the five separate calls (SURVEY 8(b) semantics)."""
        dt = self.hydro_estimate_dt()
        self.hydro_fill_ghosts(0)
        self.hydro_advance_stage(0, dt)
        self.hydro_fill_ghosts(1)
        self.hydro_advance_stage(1, dt)
        return dt

    def close(self):
        if getattr(self, "h", None) is not None and self.h:
            lib().hydro_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

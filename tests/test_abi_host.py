"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol that
include/hydro.h declares, the size queries and parameter validation work without a GPU, and
the Python struct mirrors the C struct."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2007_05218_b200 import binding as B
from paper_2007_05218_b200 import build as build_mod
from paper_2007_05218_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build_mod.build()
    return B.lib()


def test_header_symbols_all_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "hydro.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(hydro_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(B.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_probe_library_is_separate(lib):
    """The FP64-pipe probe of bench.py is a library of its own: hydro.h declares no probe, and
    hydro_probe.h's one symbol is exported by libhydro_probe_b200.so, not by the product."""
    hdr = open(os.path.join(ROOT, "include", "hydro_probe.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(hydro_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(B.PROBE_EXPORTS)
    P = B.probe_lib()
    for name in declared:
        assert hasattr(P, name) and not hasattr(lib, name)


def test_struct_layout_matches_header():
    # 3+3+1+1+3+3 int32 = 56 bytes, then 3+3+1+1+3+1+1 doubles = 104 bytes, then flatten + evolve_eint, then dx[3]
    assert C.sizeof(B.HydroParams) == 56 + 104 + 8 + 24 and B.HydroParams.flatten.offset == 160
    assert B.HydroParams.dx.offset == 168
    assert B.HydroParams.prob_lo.offset == 56 and B.HydroParams.small_pres.offset == 152


def test_size_queries_and_validation(lib):
    for n in range(1, 6):
        wl = W.config(n)
        p = B.make_params(wl.params)
        assert B.hydro_state_bytes(p) == wl.state_bytes
        assert B.hydro_scratch_bytes(p) >= wl.zones * wl.nflux * 8
    wl5 = W.config(5)
    assert wl5.state_bytes == 64 * 19 * 136 ** 3 * 8                     # 24.47 GB
    bad = W.config(3)
    bad.params["nbox"] = [60, 64, 64]
    assert B.hydro_state_bytes(B.make_params(bad.params)) == 0
    bad = W.config(3)
    bad.params["ng"] = 2
    assert B.hydro_state_bytes(B.make_params(bad.params)) == 0
    bad = W.config(3)
    bad.params["bc_hi"] = [1, 0, 0]
    assert B.hydro_state_bytes(B.make_params(bad.params)) == 0


def test_option_fields_are_validated(lib):
    ok = W.config(3)
    for key, bad in (("flatten", 2), ("flatten", -1), ("evolve_eint", 2), ("evolve_eint", -3)):
        w = W.config(3)
        w.params[key] = bad
        assert B.hydro_state_bytes(B.make_params(w.params)) == 0, (key, bad)
    w = W.config(3); w.params["flatten"] = 1; w.params["evolve_eint"] = 1
    p0, p1 = B.make_params(ok.params), B.make_params(w.params)
    assert B.hydro_state_bytes(p1) == B.hydro_state_bytes(p0)
    # flattening adds 4 padded arrays per box, the evolved energy 3 accumulator slots per zone
    extra = B.hydro_scratch_bytes(p1) - B.hydro_scratch_bytes(p0)
    assert extra >= 4 * ok.nboxes * int(np.prod(ok.nt)) * 8 + 3 * ok.zones * 8


def test_null_handle_calls_fail_cleanly(lib):
    assert lib.hydro_fill_ghosts(None, 0) == B.HYDRO_EINVAL
    assert lib.hydro_advance_stage(None, 0, 0.1) == B.HYDRO_EINVAL
    assert lib.hydro_destroy(None) == 0
    assert lib.hydro_launch_count(None) == 0
    assert isinstance(lib.hydro_last_error(None), bytes)
    out = C.c_void_p()
    p = B.make_params(W.config(1).params)
    assert lib.hydro_init(C.byref(p), None, None, None, 0, None, C.byref(out)) == B.HYDRO_EINVAL
    assert b"null device buffer" in lib.hydro_last_error(None)

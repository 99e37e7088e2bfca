"""Build step: compile csrc/hydro_api.cu into paper_2007_05218_b200/libhydro_b200.so (the product,
include/hydro.h) and csrc/fp64_probe.cu into libhydro_probe_b200.so (bench.py's FP64-pipe probe,
include/hydro_probe.h).

nvcc cross-compiles for sm_100a without a GPU.  `python -m paper_2007_05218_b200.build`
or build().  HYDRO_FMAD=0 builds with -fmad=false (every operation rounded separately, as
the scheme's definition is written); the default lets ptxas contract a*b+c into FMA.
HYDRO_NVCC_EXTRA adds nvcc flags (e.g. -DHYDRO_RING_D=6); it is part of the freshness stamp.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhydro_b200.so")
PROBE_LIB = os.path.join(HERE, "libhydro_probe_b200.so")
SOURCES = ["hydro_api.cu"]
HEADERS = ["hydro_device.cuh", "sweep_x.cuh", "sweep_xc.cuh", "sweep_yz.cuh", "march_ring.cuh", "march_x.cuh", "ctu.cuh", "amr_fill.cuh", "ghost_reduce.cuh",
           "flatten.cuh"]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo"]


def nvcc_cmd(fmad: bool, out: str = LIB, extra=()):
    return ["nvcc", "-std=c++17", "-O3", *ARCH,
            f"-fmad={'true' if fmad else 'false'}", *([] if fmad else ["-DHYDRO_STRICT"]), "-shared", "-Xcompiler", "-fPIC",
            "-o", out, *extra, *os.environ.get("HYDRO_NVCC_EXTRA", "").split(),
            *[os.path.join(CSRC, s) for s in SOURCES]]


def _run(cmd, verbose):
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose:
        sys.stderr.write(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + res.stdout + res.stderr)


def build_probe(force: bool = False, verbose: bool = False) -> str:
    src = os.path.join(CSRC, "fp64_probe.cu")
    deps = [src, os.path.join(os.path.dirname(HERE), "include", "hydro_probe.h")]
    if (not force and os.path.exists(PROBE_LIB)
            and all(os.path.getmtime(PROBE_LIB) >= os.path.getmtime(d) for d in deps)):
        return PROBE_LIB
    _run(["nvcc", "-std=c++17", "-O3", *ARCH, "-shared", "-Xcompiler", "-fPIC", "-o", PROBE_LIB, src], verbose)
    return PROBE_LIB


def build(force: bool = False, fmad=None, verbose: bool = False) -> str:
    if fmad is None:
        fmad = os.environ.get("HYDRO_FMAD", "1") != "0"
    build_probe(force=force, verbose=verbose)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [
        os.path.join(os.path.dirname(HERE), "include", "hydro.h"), os.path.abspath(__file__)]
    stamp = LIB + ".flags"
    flags = "fmad=%d extra=%s" % (int(fmad), os.environ.get("HYDRO_NVCC_EXTRA", ""))
    fresh = (os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read() == flags
             and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps))
    if fresh and not force:
        return LIB
    _run(nvcc_cmd(fmad, extra=["-Xptxas", "-v"] if verbose else []), verbose)
    with open(stamp, "w") as f:
        f.write(flags)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))

"""Compile oracle/hydro_oracle.c into oracle/liboracle_hydro.so (gcc, no FMA contraction).

Run as `python -m oracle.build_oracle` or call build().  Building the checker is not
using it: __graft_entry__.build() calls this too.

HYDRO_ORACLE_SANITIZE=1 builds and returns oracle/liboracle_hydro_san.so instead: the same source
with -fsanitize=address,undefined (out-of-bounds and use-after-free accesses, signed overflow,
misaligned or null pointers, bad shifts).  A sanitized library loaded into an unsanitized python
needs the sanitizer runtimes first in the link order, and python's own allocations are not the
oracle's leaks:

    HYDRO_ORACLE_SANITIZE=1 ASAN_OPTIONS=detect_leaks=0 UBSAN_OPTIONS=halt_on_error=1 \
    LD_PRELOAD="$(gcc -print-file-name=libasan.so) $(gcc -print-file-name=libubsan.so)" \
    python -m pytest tests -q -m "not gpu" -k oracle
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hydro_oracle.c")
LIB = os.path.join(HERE, "liboracle_hydro.so")
SAN_LIB = os.path.join(HERE, "liboracle_hydro_san.so")
FLAGS = ["-std=c99", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    sanitize = os.environ.get("HYDRO_ORACLE_SANITIZE", "0") not in ("", "0")
    lib = SAN_LIB if sanitize else LIB
    if (not force and os.path.exists(lib)
            and os.path.getmtime(lib) >= os.path.getmtime(SRC)):
        return lib
    opt = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined"] if sanitize else ["-O2"]
    subprocess.run(["gcc", *opt, *FLAGS, "-o", lib, SRC, "-lm"], check=True)
    return lib


if __name__ == "__main__":
    print(build(force=True))

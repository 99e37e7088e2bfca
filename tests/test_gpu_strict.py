"""The strict build (HYDRO_FMAD=0: -fmad=false -DHYDRO_STRICT) is the scheme's definition bit for bit: compiled
here into a temporary file and compared with the oracle with == on every valid zone after three steps, with and
without the optional O10 / O11, on ring and fallback geometries."""
import os
import subprocess
import sys
import tempfile

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_strict_build_reproduces_the_oracle_bit_for_bit():
    sys.path.insert(0, ROOT)
    from paper_2007_05218_b200 import build as build_mod
    with tempfile.TemporaryDirectory() as tmp:
        lib = os.path.join(tmp, "libhydro_b200_strict.so")
        res = subprocess.run(build_mod.nvcc_cmd(False, out=lib), capture_output=True, text=True)
        assert res.returncode == 0, res.stderr[-2000:]
        env = dict(os.environ, HYDRO_LIB=lib)
        run = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "strict_bits_helper.py")], env=env,
                             capture_output=True, text=True, timeout=900)
        assert run.returncode == 0, run.stdout[-3000:] + run.stderr[-2000:]
        assert run.stdout.count("bitwise") >= 12 and "DIFFERS" not in run.stdout

"""Hardware facts the kernels' exactness arguments rest on, measured on the GPU the tests run on.

The approximate-quotient filters (rt_bundle.cuh scan_filtered, rt_fast.cuh q_key) rule reactions
out of the argmin with q~ = (P - T) * rcp.approx.ftz.f64(a).  Their tolerances assume that the
instruction is within 2^-19.5 relative of 1/a on the range the kernels use it on; that number is
not in any PTX guarantee, so it is measured here (tests/helpers/rcp_bound.cu: > 8e9 inputs, every
exponent of the range, structured and random mantissas)."""
import os
import re
import shutil
import subprocess

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
pytestmark = pytest.mark.gpu


def test_rcp_approx_f64_error_bound(tmp_path):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not os.path.exists(nvcc):
        nvcc = shutil.which("nvcc")
    assert nvcc, "nvcc is needed to build tests/helpers/rcp_bound.cu"
    exe = str(tmp_path / "rcp_bound")
    subprocess.run([nvcc, "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-o", exe,
                    os.path.join(HERE, "helpers", "rcp_bound.cu")], check=True)
    out = subprocess.run([exe], check=True, capture_output=True, text=True, timeout=300).stdout
    m = re.search(r"inputs=(\d+) max_rel_err=(\S+)", out)
    assert m, out
    n, err = int(m.group(1)), float.fromhex(m.group(2))
    assert n > 8_000_000_000
    # scan_filtered: tolerance 2^-16 against 2^-19.5 (+ 2^-24 conversion); q_key: 32 key units
    # against 2 * (2.9 + 1) units of key error + 16 of lag (rt_fast.cuh header)
    assert 0.0 < err < 2.0 ** -19.5, out

"""Host logic of the xy FFT passes: the __host__ __device__ stage functions of csrc/fft_engine.cuh (register butterflies,
in-place digit-reversed stages, direct-global edge stage with recurrence twiddles, factorisation, twiddle tables), run
sequentially on the CPU and compared with the DFT definition in long double.  Needs nvcc, no GPU."""
import os
import shutil
import subprocess

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
SIZES = [2, 3, 4, 5, 8, 9, 15, 16, 18, 24, 25, 48, 50, 96, 108, 120, 192, 216, 240, 384, 540, 768, 1080, 2160, 4320]


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", shutil.which("nvcc")):
        if c and os.path.exists(c):
            return c
    return None


@pytest.mark.skipif(_nvcc() is None, reason="nvcc not available")
def test_fft_engine_matches_the_dft_definition(tmp_path):
    exe = str(tmp_path / "fft_engine_host")
    subprocess.check_call([_nvcc(), "-O1", "-std=c++17", "-o", exe, os.path.join(HERE, "fft_engine_host.cu")],
                          stdout=subprocess.DEVNULL, stderr=subprocess.DEVNULL)
    out = subprocess.check_output([exe] + [str(n) for n in SIZES], text=True).strip().splitlines()
    assert len(out) == len(SIZES)
    for line, n in zip(out, SIZES):
        f = line.split()
        assert int(f[0]) == n and "unsupported" not in line, line
        errs = [float(v) for v in f[1:5]]
        assert max(errs) < 2e-15, line            # forward (plain, edge), round trip (plain, edge)
        prod = 1
        for r in f[5:]:
            prod *= int(r)
        assert prod == n, line
    # sizes with a prime factor other than 2, 3, 5 are rejected (the plan then falls back to cuFFT)
    out = subprocess.check_output([exe, "14", "22", "26"], text=True)
    assert out.count("unsupported") == 3

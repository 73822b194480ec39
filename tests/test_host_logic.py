"""Host-side check of the FFT building blocks of the CUDA path (no GPU): fft_core.cuh is plain C++ on the host, so its
radix plans, stored order (pos2freq / freq2pos), staged DIF / DIT butterflies and Hermitian pair formulas are compiled
with g++ and compared with a naive DFT (tests/host/fft_core_host_check.cpp).  This is not the oracle and shares nothing
with it; it only makes a broken butterfly show up without a GPU."""
import shutil
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


def test_fft_core_on_the_host(tmp_path):
    gxx = shutil.which("g++")
    cuda_inc = Path("/usr/local/cuda/include")
    if gxx is None or not (cuda_inc / "cuda_runtime.h").exists():
        pytest.skip("needs g++ and the CUDA headers")
    exe = tmp_path / "fft_core_host_check"
    src = ROOT / "tests" / "host" / "fft_core_host_check.cpp"
    subprocess.run([gxx, "-O1", "-std=c++17", f"-I{cuda_inc}", f"-I{ROOT / 'paper_2106_03452_b200' / 'csrc'}", "-x", "c++",
                    str(src), "-o", str(exe)], check=True)
    res = subprocess.run([str(exe)], capture_output=True, text=True)
    assert res.returncode == 0 and res.stdout.strip().endswith("OK"), res.stdout + res.stderr

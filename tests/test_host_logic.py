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


def test_fused_latency_path_emulated_on_the_host(tmp_path):
    """The phase bodies of the latency path (csrc/fused_small.cuh) are __host__ __device__ templates: the whole forward
    and backward run here on the CPU, "CTA" after "CTA" between the grid barriers (tests/host/fused_emulate.cpp), and
    must match the float64 oracle within the GPU bars.  Catches tile / slot / swizzle / bin index mistakes without a
    GPU; thread-level races are of course not modelled."""
    import struct

    import numpy as np

    from oracle import dpsr_oracle as orc
    from paper_2106_03452_b200 import inputs
    gxx = shutil.which("g++")
    cuda_inc = Path("/usr/local/cuda/include")
    if gxx is None or not (cuda_inc / "cuda_runtime.h").exists():
        pytest.skip("needs g++ and the CUDA headers")
    exe = tmp_path / "fused_emulate"
    src = ROOT / "tests" / "host" / "fused_emulate.cpp"
    subprocess.run([gxx, "-O1", "-std=c++17", f"-I{cuda_inc}", f"-I{ROOT / 'paper_2106_03452_b200' / 'csrc'}", "-x", "c++",
                    str(src), "-o", str(exe)], check=True)
    for N, B, P, sigma, shape in ((32, 3, 777, 2.0, "sphere"), (64, 1, 3000, 3.0, "torus"), (128, 1, 4099, 2.0, "ellipsoids3")):
        pts = np.empty((B, P, 3), np.float32)
        nrm = np.empty((B, P, 3), np.float32)
        for b in range(B):
            pts[b], nrm[b] = inputs.make_cloud(shape, P, seed=40 + b)
        pts[0, :20, 0] = (N - 0.25) / N          # last x cell: the +1 corner wraps to plane 0
        G = inputs.upstream_grad(N, B, seed=8)
        fin, fout = tmp_path / "in.bin", tmp_path / "out.bin"
        with open(fin, "wb") as f:
            f.write(struct.pack("iiif", N, B, P, sigma))
            f.write(pts.tobytes()); f.write(nrm.tobytes()); f.write(G.tobytes())
        res = subprocess.run([str(exe), str(fin), str(fout)], capture_output=True, text=True)
        assert res.returncode == 0 and res.stdout.strip().endswith("OK"), res.stdout + res.stderr
        out = np.fromfile(fout, np.float32)
        V = N ** 3
        chi = out[:B * V].reshape(B, N, N, N)
        o = B * V + 4 * B
        gp = out[o:o + B * P * 3].reshape(B, P, 3)
        gn = out[o + B * P * 3:o + 2 * B * P * 3].reshape(B, P, 3)
        for b in range(B):
            f = orc.forward(N, sigma, pts[b], nrm[b])
            bk = orc.backward(N, sigma, pts[b], nrm[b], f, G[b])
            assert np.abs(chi[b] - f["chi"]).max() <= 1e-4 * np.abs(f["chi"]).max()
            assert np.linalg.norm(gp[b] - bk["grad_points"]) <= 1e-3 * np.linalg.norm(bk["grad_points"])
            assert np.linalg.norm(gn[b] - bk["grad_normals"]) <= 1e-3 * np.linalg.norm(bk["grad_normals"])

"""Builds libsap_dpsr.so (sm_100a only) in-tree with nvcc.  `python -m paper_2106_03452_b200.build`."""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libsap_dpsr.so"
SOURCES = [CSRC / "sap_dpsr.cu", CSRC / "sap_mesh.cu"]
HEADERS = [CSRC / "fft_core.cuh", CSRC / "zwarp_pass.cuh", CSRC / "zwarp_inv.cuh", CSRC / "fused_small.cuh", CSRC / "dpsr_kernels.cuh", CSRC / "zy_pass.cuh", CSRC / "spectral.cuh", CSRC / "ring_pass.cuh", CSRC / "zline_pass.cuh", PKG.parent / "include" / "sap_dpsr.h", PKG.parent / "include" / "sap_mesh.h"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "--expt-relaxed-constexpr", *os.environ.get("SAP_NVCC_EXTRA", "").split(), "-shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v",
]


def is_stale() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(p.stat().st_mtime > t for p in SOURCES + HEADERS + [Path(__file__)])


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not is_stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
    cmd = [nvcc, *NVCC_FLAGS, *map(str, SOURCES), "-o", str(tmp)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building libsap_dpsr.so")
    (PKG / "build_ptxas.log").write_text(res.stdout + res.stderr)
    if verbose:
        print(res.stdout + res.stderr)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))

"""ctypes loader for the float64 CPU oracle (oracle/dpsr_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It holds argument marshalling
only -- all arithmetic lives in dpsr_oracle.c, which cites the paper passage each step follows.
Nothing here imports, links or reads the CUDA package.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "dpsr_oracle.c"
_LIB = None

_dp = ctypes.POINTER(ctypes.c_double)


def _flags() -> list[str]:
    flags = ["-O3", "-fopenmp", "-shared", "-fPIC", "-std=c11", "-fno-fast-math"]
    try:
        cpu = Path("/proc/cpuinfo").read_text()
        if " avx2 " in cpu and " fma " in cpu:
            flags += ["-mavx2", "-mfma"]
    except OSError:
        pass
    return flags


def lib_path() -> Path:
    tag = hashlib.sha1((" ".join(_flags()) + _SRC.read_text()).encode()).hexdigest()[:10]
    return _HERE / f"libdpsr_oracle.{tag}.so"


def build(force: bool = False) -> Path:
    """Compile dpsr_oracle.c with gcc into oracle/libdpsr_oracle.<tag>.so (tag = flags+source hash)."""
    out = lib_path()
    if out.exists() and not force:
        return out
    for old in _HERE.glob("libdpsr_oracle.*.so"):
        try:
            old.unlink()
        except OSError:
            pass
    tmp = out.with_suffix(f".tmp{os.getpid()}")
    cmd = ["gcc", *_flags(), str(_SRC), "-o", str(tmp), "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, out)
    return out


def _load():
    global _LIB
    if _LIB is not None:
        return _LIB
    lib = ctypes.CDLL(str(build()))
    i, l, d = ctypes.c_int, ctypes.c_long, ctypes.c_double
    lib.oracle_num_threads.restype = i
    lib.oracle_splat.argtypes = [i, l, _dp, _dp, _dp, _dp]
    lib.oracle_splat.restype = None
    lib.oracle_interp.argtypes = [i, l, _dp, _dp, _dp]
    lib.oracle_interp.restype = None
    lib.oracle_dft3.argtypes = [i, _dp, _dp, _dp, _dp, i]
    lib.oracle_dft3.restype = i
    lib.oracle_dft3_direct.argtypes = [i, _dp, _dp, _dp, _dp, i]
    lib.oracle_dft3_direct.restype = None
    lib.oracle_multiplier.argtypes = [i, d, i, i, i, _dp]
    lib.oracle_multiplier.restype = None
    lib.oracle_spectral_solve.argtypes = [i, d, _dp, _dp, _dp, _dp]
    lib.oracle_spectral_solve.restype = None
    lib.oracle_spectral_adjoint.argtypes = [i, d, _dp, _dp, _dp, _dp]
    lib.oracle_spectral_adjoint.restype = None
    lib.oracle_dpsr_forward.argtypes = [i, d, l, _dp, _dp, _dp, _dp, _dp, _dp, _dp]
    lib.oracle_dpsr_forward.restype = i
    lib.oracle_dpsr_backward.argtypes = [i, d, l, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp]
    lib.oracle_dpsr_backward.restype = i
    lib.oracle_chi_tilde_at.argtypes = [i, d, l, _dp, _dp, i, i, i, _dp]
    lib.oracle_chi_tilde_at.restype = None
    _LIB = lib
    return lib


def _c(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def splat(N, points, normals):
    """Eq.10-11.  Returns (v [3,N,N,N], W [N,N,N])."""
    pts, nrm = _c(points), _c(normals)
    P = pts.shape[0]
    assert pts.shape == (P, 3) and nrm.shape == (P, 3)
    v = np.empty((3, N, N, N))
    W = np.empty((N, N, N))
    _load().oracle_splat(N, P, _p(pts), _p(nrm), _p(v), _p(W))
    return v, W


def interp(N, points, grid):
    pts, g = _c(points), _c(grid, (N, N, N))
    out = np.empty(pts.shape[0])
    _load().oracle_interp(N, pts.shape[0], _p(pts), _p(g), _p(out))
    return out


def dft3(x, sign=-1, direct=False):
    """Naive 3-D DFT of a cubic array (complex or real).  sign=-1 forward, +1 inverse (1/N^3)."""
    x = np.asarray(x)
    N = x.shape[0]
    assert x.shape == (N, N, N)
    re = _c(x.real)
    im = _c(x.imag) if np.iscomplexobj(x) else None
    ore, oim = np.empty((N, N, N)), np.empty((N, N, N))
    lib = _load()
    if direct:
        lib.oracle_dft3_direct(N, _p(re), _p(im), _p(ore), _p(oim), sign)
    else:
        rc = lib.oracle_dft3(N, _p(re), _p(im), _p(ore), _p(oim), sign)
        if rc:
            raise MemoryError("oracle_dft3")
    return ore + 1j * oim


def multiplier(N, sigma, kx, ky, kz):
    """Real m_c with M_c(k) = i m_c(k) (Eq.3 with readings R3/R4/R6)."""
    m = np.empty(3)
    _load().oracle_multiplier(N, float(sigma), kx, ky, kz, _p(m))
    return m


def spectral_solve(N, sigma, vt):
    """vt: complex [3,N,N,N] -> chi~ complex [N,N,N] (Eq.3)."""
    vt = np.asarray(vt)
    re, im = _c(vt.real, (3, N, N, N)), _c(vt.imag, (3, N, N, N))
    ore, oim = np.empty((N, N, N)), np.empty((N, N, N))
    _load().oracle_spectral_solve(N, float(sigma), _p(re), _p(im), _p(ore), _p(oim))
    return ore + 1j * oim


def spectral_adjoint(N, sigma, gt):
    gt = np.asarray(gt)
    re, im = _c(gt.real, (N, N, N)), _c(gt.imag, (N, N, N))
    ore, oim = np.empty((3, N, N, N)), np.empty((3, N, N, N))
    _load().oracle_spectral_adjoint(N, float(sigma), _p(re), _p(im), _p(ore), _p(oim))
    return ore + 1j * oim


def forward(N, sigma, points, normals, intermediates=False):
    """DPSR forward (Eq.2-4).  Returns dict(chi, mu, a, s, imag_residue[, chi_prime, v, W])."""
    pts, nrm = _c(points), _c(normals)
    P = pts.shape[0]
    assert pts.shape == (P, 3) and nrm.shape == (P, 3)
    chi = np.empty((N, N, N))
    cp = np.empty((N, N, N))
    W = np.empty((N, N, N))
    v = np.empty((3, N, N, N)) if intermediates else None
    stats = np.empty(4)
    rc = _load().oracle_dpsr_forward(N, float(sigma), P, _p(pts), _p(nrm), _p(chi), _p(cp),
                                     _p(v), _p(W), _p(stats))
    if rc:
        raise RuntimeError(f"oracle_dpsr_forward rc={rc}")
    out = dict(chi=chi, chi_prime=cp, W=W, mu=stats[0], a=stats[1], s=stats[2],
               imag_residue=stats[3])
    if intermediates:
        out["v"] = v
    return out


def backward(N, sigma, points, normals, fwd, G, intermediates=False):
    """Exact adjoint.  fwd = the dict returned by forward().  Returns dict(grad_points, grad_normals[, gbar, vbar])."""
    pts, nrm = _c(points), _c(normals)
    P = pts.shape[0]
    cp, W, G = _c(fwd["chi_prime"], (N, N, N)), _c(fwd["W"], (N, N, N)), _c(G, (N, N, N))
    stats = np.array([fwd["mu"], fwd["a"], fwd["s"]], dtype=np.float64)
    gp, gn = np.empty((P, 3)), np.empty((P, 3))
    gbar = np.empty((N, N, N)) if intermediates else None
    vbar = np.empty((3, N, N, N)) if intermediates else None
    rc = _load().oracle_dpsr_backward(N, float(sigma), P, _p(pts), _p(nrm), _p(cp), _p(W),
                                      _p(stats), _p(G), _p(gp), _p(gn), _p(gbar), _p(vbar))
    if rc:
        raise RuntimeError(f"oracle_dpsr_backward rc={rc}")
    out = dict(grad_points=gp, grad_normals=gn)
    if intermediates:
        out.update(gbar=gbar, vbar=vbar)
    return out


def chi_tilde_at(N, sigma, points, normals, k):
    """One coefficient chi~(k) of the unnormalised chi' computed straight from the points, O(8P)."""
    pts, nrm = _c(points), _c(normals)
    out = np.empty(2)
    _load().oracle_chi_tilde_at(N, float(sigma), pts.shape[0], _p(pts), _p(nrm),
                                int(k[0]), int(k[1]), int(k[2]), _p(out))
    return complex(out[0], out[1])

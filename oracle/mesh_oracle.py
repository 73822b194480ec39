"""ctypes loader for the float64 CPU oracle of the mesh side of the pipeline (oracle/mesh_oracle.c): Marching Cubes
(PAPER.md:L100), the surrogate gradient of Eq.6 (L113-L117) and the bi-directional L2 Chamfer distance (L102).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import
this module.  Argument marshalling only -- the arithmetic lives in mesh_oracle.c.  Nothing here imports, links or reads
the CUDA package.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "mesh_oracle.c"
_LIB = None
MC_MAX_TRI = 12

_dp = ctypes.POINTER(ctypes.c_double)
_lp = ctypes.POINTER(ctypes.c_long)
_ip = ctypes.POINTER(ctypes.c_int)
_FLAGS = ["-O2", "-shared", "-fPIC", "-std=c11", "-fno-fast-math"]


def lib_path() -> Path:
    tag = hashlib.sha1((" ".join(_FLAGS) + _SRC.read_text()).encode()).hexdigest()[:10]
    return _HERE / f"libmesh_oracle.{tag}.so"


def build(force: bool = False) -> Path:
    out = lib_path()
    if out.exists() and not force:
        return out
    for old in _HERE.glob("libmesh_oracle.*.so"):
        try:
            old.unlink()
        except OSError:
            pass
    tmp = out.with_suffix(f".tmp{os.getpid()}")
    subprocess.run(["gcc", *_FLAGS, str(_SRC), "-o", str(tmp), "-lm"], check=True)
    os.replace(tmp, out)
    return out


def _load():
    global _LIB
    if _LIB is not None:
        return _LIB
    lib = ctypes.CDLL(str(build()))
    i, l = ctypes.c_int, ctypes.c_long
    lib.mesh_oracle_mc_table.argtypes = [_ip, _ip]
    lib.mesh_oracle_mc_table.restype = i
    lib.mesh_oracle_mc_count.argtypes = [i, _dp, _lp, _lp]
    lib.mesh_oracle_mc_count.restype = None
    lib.mesh_oracle_mc_extract.argtypes = [i, _dp, _dp, _dp, _lp, _ip, _dp, _lp]
    lib.mesh_oracle_mc_extract.restype = None
    lib.mesh_oracle_eq6_backward.argtypes = [i, l, _lp, _ip, _dp, _dp, _dp, _dp]
    lib.mesh_oracle_eq6_backward.restype = None
    lib.mesh_oracle_chamfer.argtypes = [l, _dp, l, _dp, _lp, _lp, _dp, _dp, _dp, _dp, _dp]
    lib.mesh_oracle_chamfer.restype = None
    _LIB = lib
    return lib


def _d(a):
    return a.ctypes.data_as(_dp)


def _l(a):
    return a.ctypes.data_as(_lp)


def _i(a):
    return a.ctypes.data_as(_ip)


def mc_table():
    """(ntri[256], tris[256, 12, 3]) of cube-edge ids, -1 padded: the triangulation rule M3 for every sign configuration."""
    ntri = np.zeros(256, np.int32)
    tris = np.zeros((256, MC_MAX_TRI, 3), np.int32)
    _load().mesh_oracle_mc_table(_i(ntri), _i(tris))
    return ntri, tris


def marching_cubes(chi):
    """chi: [N,N,N] (any float dtype, promoted to float64).  Returns dict(verts [V,3] in the unit cube, normals [V,3],
    tris [T,3] vertex ids, vnode [V], vaxis [V], vt [V])."""
    chi = np.ascontiguousarray(chi, dtype=np.float64)
    N = chi.shape[0]
    assert chi.shape == (N, N, N)
    nv, nt = ctypes.c_long(), ctypes.c_long()
    lib = _load()
    lib.mesh_oracle_mc_count(N, _d(chi), ctypes.byref(nv), ctypes.byref(nt))
    V, T = nv.value, nt.value
    verts = np.zeros((V, 3)); normals = np.zeros((V, 3))
    vnode = np.zeros(V, np.int64); vaxis = np.zeros(V, np.int32); vt = np.zeros(V)
    tris = np.zeros((T, 3), np.int64)
    lib.mesh_oracle_mc_extract(N, _d(chi), _d(verts), _d(normals), _l(vnode), _i(vaxis), _d(vt), _l(tris))
    return dict(verts=verts, normals=normals, tris=tris, vnode=vnode, vaxis=vaxis, vt=vt)


def eq6_backward(N, mesh, dLdp):
    """G [N,N,N] = dL/dchi from dL/dp_mesh [V,3] through Eq.6 (reading M5)."""
    dLdp = np.ascontiguousarray(dLdp, dtype=np.float64)
    V = mesh["verts"].shape[0]
    assert dLdp.shape == (V, 3)
    G = np.zeros((N, N, N))
    _load().mesh_oracle_eq6_backward(N, V, _l(mesh["vnode"]), _i(mesh["vaxis"]), _d(mesh["vt"]),
                                     _d(np.ascontiguousarray(mesh["normals"])), _d(dLdp), _d(G))
    return G


def chamfer(a, b, grads=True):
    """Bi-directional squared-L2 Chamfer distance (M6) between point sets a [na,3] and b [nb,3], brute force."""
    a = np.ascontiguousarray(a, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    na, nb = a.shape[0], b.shape[0]
    nn_a = np.zeros(na, np.int64); nn_b = np.zeros(nb, np.int64)
    da = np.zeros(na); db = np.zeros(nb)
    loss = ctypes.c_double()
    ga = np.zeros((na, 3)); gb = np.zeros((nb, 3))
    _load().mesh_oracle_chamfer(na, _d(a), nb, _d(b), _l(nn_a), _l(nn_b), _d(da), _d(db), ctypes.byref(loss),
                                _d(ga) if grads else None, _d(gb) if grads else None)
    return dict(loss=loss.value, nn_a=nn_a, nn_b=nn_b, dist_a=da, dist_b=db, grad_a=ga, grad_b=gb)

"""Thin ctypes binding of the mesh entry points of libsap_dpsr.so (include/sap_mesh.h): Marching Cubes on the
indicator grid, the surrogate gradient of Eq.6 and the bi-directional L2 Chamfer distance (Sec.3.2,
L96-L121).  Argument marshalling only; every step runs in the library's CUDA kernels.  No fallback."""
from __future__ import annotations

import ctypes

from .binding import SAP_OK, SapError, _stream_ptr, lib as _dpsr_lib

EXPORTS = ["sap_mesh_create", "sap_mc_extract", "sap_mc_backward", "sap_chamfer", "sap_mc_table", "sap_mesh_destroy",
           "sap_mesh_last_error", "sap_mesh_workspace_bytes", "sap_mesh_last_launch_count", "sap_points_sgd_step", "sap_chamfer_set_search",
           "sap_chamfer_nn_static"]
MC_MAX_TRI = 12
NN_STATIC_MAX_QUERIES = 262144   # SAP_NN_STATIC_MAX_QUERIES of include/sap_mesh.h
_ready = False


def lib():
    global _ready
    L = _dpsr_lib()
    if not _ready:
        vp, ci = ctypes.c_void_p, ctypes.c_int
        L.sap_mesh_create.argtypes = [ci, ci, ci, ci, ctypes.POINTER(vp)]
        L.sap_mesh_create.restype = ci
        L.sap_mc_extract.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.sap_mc_extract.restype = ci
        L.sap_mc_backward.argtypes = [vp, vp, vp, vp, vp]
        L.sap_mc_backward.restype = ci
        L.sap_chamfer.argtypes = [vp, vp, ci, vp, vp, ci, vp, vp, vp, vp, vp]
        L.sap_chamfer.restype = ci
        L.sap_mc_table.argtypes = [vp, vp]
        L.sap_mc_table.restype = ci
        L.sap_points_sgd_step.argtypes = [vp, vp, vp, vp, ci, ci, ctypes.c_float, vp, vp]
        L.sap_points_sgd_step.restype = ci
        L.sap_chamfer_set_search.argtypes = [vp, ci]
        L.sap_chamfer_set_search.restype = ci
        L.sap_chamfer_nn_static.argtypes = [vp, ci, vp, ci, vp, vp, vp]
        L.sap_chamfer_nn_static.restype = ci
        L.sap_mesh_destroy.argtypes = [vp]
        L.sap_mesh_destroy.restype = None
        L.sap_mesh_last_error.argtypes = [vp]
        L.sap_mesh_last_error.restype = ctypes.c_char_p
        L.sap_mesh_workspace_bytes.argtypes = [vp]
        L.sap_mesh_workspace_bytes.restype = ctypes.c_size_t
        L.sap_mesh_last_launch_count.argtypes = [vp]
        L.sap_mesh_last_launch_count.restype = ci
        _ready = True
    return L


def mc_table():
    """(ntri[256], tris[256, 12, 3]) cube-edge ids of the triangulation rule the library built at load (host only)."""
    import numpy as np
    ntri = np.zeros(256, np.int32)
    tris = np.zeros((256, MC_MAX_TRI, 3), np.int32)
    lib().sap_mc_table(ntri.ctypes.data_as(ctypes.c_void_p), tris.ctypes.data_as(ctypes.c_void_p))
    return ntri, tris


def sgd_step(points, normals, grad_points, grad_normals, N, move, scratch, stream=None):
    """sap_points_sgd_step on CUDA float32 tensors of equal size (in place); scratch: CUDA int32/uint32 tensor [1]."""
    st = lib().sap_points_sgd_step(ctypes.c_void_p(points.data_ptr()), ctypes.c_void_p(normals.data_ptr()),
                                   ctypes.c_void_p(grad_points.data_ptr()), ctypes.c_void_p(grad_normals.data_ptr()),
                                   int(points.numel()), int(N), float(move), ctypes.c_void_p(scratch.data_ptr()), _stream_ptr(stream))
    if st != SAP_OK:
        raise SapError(st, "sap_points_sgd_step")


def nn_static(queries, targets, nn, d2, stream=None):
    """sap_chamfer_nn_static: exact nearest target of every query (CUDA float32 [nq,3] / [nt,3], contiguous) into the
    caller's nn (int32 [nq]) and d2 (float32 [nq]).  No handle, no allocation on either side of the ABI: the scratch is the
    library's static device array (at most NN_STATIC_MAX_QUERIES queries; calls that overlap on the GPU race on it)."""
    import torch
    nq, nt = int(queries.shape[0]), int(targets.shape[0])
    for t, dt, shape, name in ((queries, torch.float32, (nq, 3), "queries"), (targets, torch.float32, (nt, 3), "targets"),
                               (nn, torch.int32, (nq,), "nn"), (d2, torch.float32, (nq,), "d2")):
        if not (t.is_cuda and t.dtype == dt and tuple(t.shape) == shape and t.is_contiguous()):
            raise ValueError(f"{name}: expected a contiguous CUDA {dt} tensor of shape {shape}")
    L = lib()
    st = L.sap_chamfer_nn_static(ctypes.c_void_p(queries.data_ptr()), nq, ctypes.c_void_p(targets.data_ptr()), nt,
                                 ctypes.c_void_p(nn.data_ptr()), ctypes.c_void_p(d2.data_ptr()), _stream_ptr(stream))
    if st != SAP_OK:
        raise SapError(st, (L.sap_mesh_last_error(None) or b"sap_chamfer_nn_static").decode())


class Mesh:
    """One handle: sap_mesh_create(N, max_vertices, max_triangles, max_points)."""

    def __init__(self, N, max_vertices, max_triangles, max_points):
        self._h = ctypes.c_void_p()
        self.N, self.max_v, self.max_t, self.max_p = int(N), int(max_vertices), int(max_triangles), int(max_points)
        L = lib()
        st = L.sap_mesh_create(self.N, self.max_v, self.max_t, self.max_p, ctypes.byref(self._h))
        if st != SAP_OK:
            self._h = ctypes.c_void_p()
            raise SapError(st, L.sap_mesh_last_error(None).decode())

    def _check(self, st):
        if st != SAP_OK:
            raise SapError(st, lib().sap_mesh_last_error(self._h).decode())

    @staticmethod
    def _p(t, dtype, shape, name):
        if not (t.is_cuda and t.dtype == dtype and t.is_contiguous() and tuple(t.shape) == tuple(shape)):
            raise ValueError(f"{name}: need a contiguous {dtype} CUDA tensor of shape {tuple(shape)}, got {tuple(t.shape)} {t.dtype}")
        return ctypes.c_void_p(t.data_ptr())

    def extract(self, chi, verts=None, normals=None, tris=None, counts=None, stream=None):
        """chi CUDA float32 [N,N,N] -> (verts [max_v,3], normals [max_v,3], tris [max_t,3] int32, counts [2] int32 = {V, T});
        rows beyond V / T are unspecified.  Nothing is synchronised."""
        import torch
        N, dev = self.N, chi.device
        verts = torch.empty((self.max_v, 3), dtype=torch.float32, device=dev) if verts is None else verts
        normals = torch.empty((self.max_v, 3), dtype=torch.float32, device=dev) if normals is None else normals
        tris = torch.empty((self.max_t, 3), dtype=torch.int32, device=dev) if tris is None else tris
        counts = torch.empty((2,), dtype=torch.int32, device=dev) if counts is None else counts
        self._check(lib().sap_mc_extract(
            self._h, self._p(chi, torch.float32, (N, N, N), "chi"), self._p(verts, torch.float32, (self.max_v, 3), "verts"),
            self._p(normals, torch.float32, (self.max_v, 3), "normals"), self._p(tris, torch.int32, (self.max_t, 3), "tris"),
            self._p(counts, torch.int32, (2,), "counts"), _stream_ptr(stream)))
        return verts, normals, tris, counts

    def backward(self, grad_verts, normals, grad_chi=None, stream=None):
        """Eq.6: dL/dp_mesh [max_v,3] -> dL/dchi [N,N,N]."""
        import torch
        N = self.N
        grad_chi = torch.empty((N, N, N), dtype=torch.float32, device=grad_verts.device) if grad_chi is None else grad_chi
        self._check(lib().sap_mc_backward(
            self._h, self._p(grad_verts, torch.float32, (self.max_v, 3), "grad_verts"),
            self._p(normals, torch.float32, (self.max_v, 3), "normals"), self._p(grad_chi, torch.float32, (N, N, N), "grad_chi"),
            _stream_ptr(stream)))
        return grad_chi

    def chamfer(self, a, b, na=None, na_dev=None, want_grad=True, want_nn=False, loss=None, grad_a=None, stream=None):
        """Bi-directional squared-L2 Chamfer distance between a [>=na,3] and b [nb,3] (CUDA float32).  na_dev: optional
        CUDA int32 tensor whose first element is the number of points of a (e.g. counts of extract).  Returns
        (loss [1], grad_a or None, nn_a or None, nn_b or None)."""
        import torch
        dev = a.device
        cap = int(a.shape[0]) if na is None else int(na)
        nb = int(b.shape[0])
        loss = torch.empty((1,), dtype=torch.float32, device=dev) if loss is None else loss
        if want_grad and grad_a is None:
            grad_a = torch.empty_like(a)
        nn_a = torch.empty((a.shape[0],), dtype=torch.int32, device=dev) if want_nn else None
        nn_b = torch.empty((nb,), dtype=torch.int32, device=dev) if want_nn else None
        null = ctypes.c_void_p()
        self._check(lib().sap_chamfer(
            self._h, self._p(a, torch.float32, a.shape, "a"), cap,
            null if na_dev is None else ctypes.c_void_p(na_dev.data_ptr()),
            self._p(b, torch.float32, (nb, 3), "b"), nb, self._p(loss, torch.float32, (1,), "loss"),
            null if grad_a is None else self._p(grad_a, torch.float32, a.shape, "grad_a"),
            null if nn_a is None else ctypes.c_void_p(nn_a.data_ptr()),
            null if nn_b is None else ctypes.c_void_p(nn_b.data_ptr()), _stream_ptr(stream)))
        return loss, grad_a, nn_a, nn_b

    def set_search(self, mode):
        """'auto' | 'brute' | 'grid': nearest-neighbour search of chamfer (include/sap_mesh.h, SAP_NN_*)."""
        self._check(lib().sap_chamfer_set_search(self._h, {"auto": 0, "brute": 1, "grid": 2}[mode]))

    @property
    def workspace_bytes(self):
        return int(lib().sap_mesh_workspace_bytes(self._h))

    @property
    def last_launch_count(self):
        return int(lib().sap_mesh_last_launch_count(self._h))

    def close(self):
        if self._h:
            lib().sap_mesh_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

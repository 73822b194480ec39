"""Thin ctypes binding of libsap_dpsr.so (include/sap_dpsr.h).  Argument marshalling only: every step
of the DPSR path (Sec.3.1, Eq.2-4; Suppl. A) runs in the library's CUDA kernels.  PyTorch is
used for device memory and streams.  There is no fallback: a missing library raises."""
from __future__ import annotations

import ctypes
from pathlib import Path

PKG = Path(__file__).resolve().parent
LIB_PATH = PKG / "libsap_dpsr.so"

SAP_OK, SAP_ERR_INVALID_ARG, SAP_ERR_UNSUPPORTED, SAP_ERR_OOM, SAP_ERR_CUDA = range(5)
STATUS_NAMES = {0: "SAP_OK", 1: "SAP_ERR_INVALID_ARG", 2: "SAP_ERR_UNSUPPORTED", 3: "SAP_ERR_OOM", 4: "SAP_ERR_CUDA"}

EXPORTS = [
    "sap_dpsr_create", "sap_dpsr_forward", "sap_dpsr_backward", "sap_dpsr_forward_mse", "sap_dpsr_backward_mse", "sap_dpsr_forward_host",
    "sap_dpsr_backward_host", "sap_dpsr_get_stats", "sap_dpsr_destroy", "sap_dpsr_last_error",
    "sap_dpsr_workspace_bytes", "sap_dpsr_last_launch_count", "sap_dpsr_set_profiling", "sap_dpsr_get_profile",
    "sap_dpsr_epoch", "sap_dpsr_check_epoch", "sap_dpsr_reserve", "sap_dpsr_set_path", "sap_dpsr_get_path",
    "sap_dpsr_get_fused_phases", "sap_dpsr_set_sparse", "sap_dpsr_get_activity",
]
SAP_PATH_AUTO, SAP_PATH_THROUGHPUT, SAP_PATH_LATENCY = 0, 1, 2
PATHS = {"auto": 0, "throughput": 1, "latency": 2}
SAP_RESERVE_MSE, SAP_RESERVE_HOST = 1, 2

_lib = None


class SapError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {msg}")
        self.status = status


def lib():
    """Loads libsap_dpsr.so (built in-tree by paper_2106_03452_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise FileNotFoundError(
            f"{LIB_PATH} not found: build it with `python -m paper_2106_03452_b200.build` "
            "(there is no CPU fallback for the DPSR path)")
    L = ctypes.CDLL(str(LIB_PATH))
    vp, ci, cf = ctypes.c_void_p, ctypes.c_int, ctypes.c_float
    L.sap_dpsr_create.argtypes = [ci, cf, ci, ci, ctypes.POINTER(vp)]
    L.sap_dpsr_create.restype = ci
    L.sap_dpsr_forward.argtypes = [vp, vp, vp, ci, vp, vp]
    L.sap_dpsr_forward.restype = ci
    L.sap_dpsr_backward.argtypes = [vp, vp, vp, ci, vp, vp, vp, vp, vp]
    L.sap_dpsr_backward.restype = ci
    L.sap_dpsr_forward_mse.argtypes = [vp, vp, vp, ci, vp, vp, vp, vp]
    L.sap_dpsr_forward_mse.restype = ci
    L.sap_dpsr_backward_mse.argtypes = [vp, vp, vp, ci, vp, vp, vp, vp]
    L.sap_dpsr_backward_mse.restype = ci
    L.sap_dpsr_forward_host.argtypes = [vp, vp, vp, ci, vp, vp]
    L.sap_dpsr_forward_host.restype = ci
    L.sap_dpsr_backward_host.argtypes = [vp, vp, vp, vp, vp]
    L.sap_dpsr_backward_host.restype = ci
    L.sap_dpsr_get_stats.argtypes = [vp, vp, vp]
    L.sap_dpsr_get_stats.restype = ci
    L.sap_dpsr_destroy.argtypes = [vp]
    L.sap_dpsr_destroy.restype = None
    L.sap_dpsr_last_error.argtypes = [vp]
    L.sap_dpsr_last_error.restype = ctypes.c_char_p
    L.sap_dpsr_workspace_bytes.argtypes = [vp]
    L.sap_dpsr_workspace_bytes.restype = ctypes.c_size_t
    L.sap_dpsr_set_sparse.argtypes = [vp, ci]
    L.sap_dpsr_set_sparse.restype = ci
    L.sap_dpsr_get_activity.argtypes = [vp, vp, vp]
    L.sap_dpsr_get_activity.restype = ci
    L.sap_dpsr_last_launch_count.argtypes = [vp]
    L.sap_dpsr_last_launch_count.restype = ci
    L.sap_dpsr_set_profiling.argtypes = [vp, ci]
    L.sap_dpsr_set_profiling.restype = ci
    L.sap_dpsr_get_profile.argtypes = [vp, ctypes.POINTER(cf), ctypes.POINTER(ctypes.c_char_p), ci]
    L.sap_dpsr_get_profile.restype = ci
    L.sap_dpsr_epoch.argtypes = [vp]
    L.sap_dpsr_epoch.restype = ctypes.c_ulonglong
    L.sap_dpsr_check_epoch.argtypes = [vp, ctypes.c_ulonglong]
    L.sap_dpsr_check_epoch.restype = ci
    L.sap_dpsr_reserve.argtypes = [vp, ci]
    L.sap_dpsr_reserve.restype = ci
    L.sap_dpsr_set_path.argtypes = [vp, ci]
    L.sap_dpsr_set_path.restype = ci
    L.sap_dpsr_get_path.argtypes = [vp]
    L.sap_dpsr_get_path.restype = ci
    L.sap_dpsr_get_fused_phases.argtypes = [vp, ctypes.POINTER(cf), ctypes.POINTER(ctypes.c_char_p), ci]
    L.sap_dpsr_get_fused_phases.restype = ci
    _lib = L
    return L


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


class Dpsr:
    """One solver handle: sap_dpsr_create(N, sigma, batch, max_points) / forward / backward / destroy."""

    def __init__(self, N, sigma, batch=1, max_points=1):
        self._h = ctypes.c_void_p()
        self.N, self.sigma, self.batch, self.max_points = int(N), float(sigma), int(batch), int(max_points)
        L = lib()
        st = L.sap_dpsr_create(self.N, self.sigma, self.batch, self.max_points, ctypes.byref(self._h))
        if st != SAP_OK:
            self._h = ctypes.c_void_p()
            raise SapError(st, L.sap_dpsr_last_error(None).decode())

    def _check(self, st):
        if st != SAP_OK:
            raise SapError(st, lib().sap_dpsr_last_error(self._h).decode())

    def _dev(self, t, shape, name):
        import torch
        if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and tuple(t.shape) == tuple(shape)):
            raise ValueError(f"{name}: need a contiguous float32 CUDA tensor of shape {tuple(shape)}, got "
                             f"{tuple(t.shape)} {t.dtype} {t.device}")
        return ctypes.c_void_p(t.data_ptr())

    def forward(self, points, normals, chi=None, stream=None):
        """points, normals: CUDA float32 [batch, P, 3] -> chi CUDA float32 [batch, N, N, N]."""
        import torch
        B, N = self.batch, self.N
        P = int(points.shape[1])
        if chi is None:
            chi = torch.empty((B, N, N, N), dtype=torch.float32, device=points.device)
        self._check(lib().sap_dpsr_forward(self._h, self._dev(points, (B, P, 3), "points"),
                                           self._dev(normals, (B, P, 3), "normals"), P,
                                           self._dev(chi, (B, N, N, N), "chi"), _stream_ptr(stream)))
        return chi

    def backward(self, points, normals, chi, grad_chi, grad_points=None, grad_normals=None, stream=None):
        import torch
        B, N = self.batch, self.N
        P = int(points.shape[1])
        if grad_points is None:
            grad_points = torch.empty_like(points)
        if grad_normals is None:
            grad_normals = torch.empty_like(normals)
        self._check(lib().sap_dpsr_backward(
            self._h, self._dev(points, (B, P, 3), "points"), self._dev(normals, (B, P, 3), "normals"), P,
            self._dev(chi, (B, N, N, N), "chi"), self._dev(grad_chi, (B, N, N, N), "grad_chi"),
            self._dev(grad_points, (B, P, 3), "grad_points"), self._dev(grad_normals, (B, P, 3), "grad_normals"),
            _stream_ptr(stream)))
        return grad_points, grad_normals

    def forward_mse(self, points, normals, chi_gt, chi=None, loss=None, stream=None):
        """Forward with the fused loss of Eq.9: returns (chi [batch,N,N,N], loss [batch] = ||chi - chi_gt||^2)."""
        import torch
        B, N = self.batch, self.N
        P = int(points.shape[1])
        if chi is None:
            chi = torch.empty((B, N, N, N), dtype=torch.float32, device=points.device)
        if loss is None:
            loss = torch.empty((B,), dtype=torch.float32, device=points.device)
        self._check(lib().sap_dpsr_forward_mse(
            self._h, self._dev(points, (B, P, 3), "points"), self._dev(normals, (B, P, 3), "normals"), P,
            self._dev(chi_gt, (B, N, N, N), "chi_gt"), self._dev(chi, (B, N, N, N), "chi"), self._dev(loss, (B,), "loss"),
            _stream_ptr(stream)))
        return chi, loss

    def backward_mse(self, points, normals, chi, grad_points=None, grad_normals=None, stream=None):
        """Gradients of the loss of the preceding forward_mse (dL/dchi is kept inside the handle)."""
        import torch
        B, N = self.batch, self.N
        P = int(points.shape[1])
        if grad_points is None:
            grad_points = torch.empty_like(points)
        if grad_normals is None:
            grad_normals = torch.empty_like(normals)
        self._check(lib().sap_dpsr_backward_mse(
            self._h, self._dev(points, (B, P, 3), "points"), self._dev(normals, (B, P, 3), "normals"), P,
            self._dev(chi, (B, N, N, N), "chi"), self._dev(grad_points, (B, P, 3), "grad_points"),
            self._dev(grad_normals, (B, P, 3), "grad_normals"), _stream_ptr(stream)))
        return grad_points, grad_normals

    @staticmethod
    def _host(t, shape, name):
        import torch
        if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() or tuple(t.shape) != tuple(shape):
            raise ValueError(f"{name}: need a contiguous float32 CPU tensor of shape {tuple(shape)}")
        return ctypes.c_void_p(t.data_ptr())

    def forward_host(self, points, normals, chi=None, stream=None):
        """Host tensors in, host chi out (chi may be None to keep it on the device only)."""
        B, N = self.batch, self.N
        P = int(points.shape[1])
        chi_p = ctypes.c_void_p() if chi is None else self._host(chi, (B, N, N, N), "chi")
        self._check(lib().sap_dpsr_forward_host(self._h, self._host(points, (B, P, 3), "points"),
                                                self._host(normals, (B, P, 3), "normals"), P, chi_p,
                                                _stream_ptr(stream)))
        return chi

    def backward_host(self, grad_chi, grad_points, grad_normals, stream=None):
        B, N = self.batch, self.N
        P = int(grad_points.shape[1])
        self._check(lib().sap_dpsr_backward_host(self._h, self._host(grad_chi, (B, N, N, N), "grad_chi"),
                                                 self._host(grad_points, (B, P, 3), "grad_points"),
                                                 self._host(grad_normals, (B, P, 3), "grad_normals"),
                                                 _stream_ptr(stream)))
        return grad_points, grad_normals

    def stats(self, stream=None):
        """[batch, 3] = (mu, a, s) of the last forward (Eq.4)."""
        import numpy as np
        out = np.empty((self.batch, 3), np.float32)
        self._check(lib().sap_dpsr_get_stats(self._h, out.ctypes.data_as(ctypes.c_void_p), _stream_ptr(stream)))
        return out

    def set_sparse(self, on=True):
        """Activity lists on / off (sap_dpsr_set_sparse); takes effect at the next forward."""
        self._check(lib().sap_dpsr_set_sparse(self._h, 1 if on else 0))

    def activity(self, stream=None):
        """(active tiles, tiles, active planes, planes) of the last throughput-path forward, summed over the batch."""
        import numpy as np
        out = np.zeros(4, np.int32)
        self._check(lib().sap_dpsr_get_activity(self._h, out.ctypes.data_as(ctypes.c_void_p), _stream_ptr(stream)))
        return tuple(int(v) for v in out)

    @property
    def epoch(self):
        """Epoch of the last forward on this handle (every forward variant increments it)."""
        return int(lib().sap_dpsr_epoch(self._h))

    def check_epoch(self, epoch):
        """Raises if another forward has run on the handle since the one that returned `epoch`."""
        self._check(lib().sap_dpsr_check_epoch(self._h, int(epoch)))

    def reserve(self, mse=False, host=False):
        """Allocates the optional buffers of the fused-loss / host-buffer entry points up front."""
        self._check(lib().sap_dpsr_reserve(self._h, (SAP_RESERVE_MSE if mse else 0) | (SAP_RESERVE_HOST if host else 0)))

    def set_path(self, path):
        """'auto' | 'throughput' | 'latency' (include/sap_dpsr.h, SAP_PATH_*)."""
        self._check(lib().sap_dpsr_set_path(self._h, PATHS[path] if isinstance(path, str) else int(path)))

    @property
    def path(self):
        return {1: "throughput", 2: "latency"}.get(int(lib().sap_dpsr_get_path(self._h)), "?")

    def fused_phases(self):
        """[(phase label, microseconds)] between the grid barriers of the last latency-path forward / backward."""
        cap = 64
        us = (ctypes.c_float * cap)()
        names = (ctypes.c_char_p * cap)()
        n = lib().sap_dpsr_get_fused_phases(self._h, us, names, cap)
        return [(names[i].decode(), float(us[i])) for i in range(n)]

    def set_profiling(self, on=True):
        self._check(lib().sap_dpsr_set_profiling(self._h, int(bool(on))))

    def profile(self):
        """[(kernel label, ms)] of the launches of the last forward or backward call (profiling on)."""
        cap = 24
        ms = (ctypes.c_float * cap)()
        names = (ctypes.c_char_p * cap)()
        n = lib().sap_dpsr_get_profile(self._h, ms, names, cap)
        return [(names[i].decode(), float(ms[i])) for i in range(n)]

    @property
    def workspace_bytes(self):
        return int(lib().sap_dpsr_workspace_bytes(self._h))

    @property
    def last_launch_count(self):
        return int(lib().sap_dpsr_last_launch_count(self._h))

    def close(self):
        if self._h:
            lib().sap_dpsr_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class DpsrFunction:
    """torch.autograd.Function factory bound to a handle: chi = apply(points, normals)."""

    @staticmethod
    def make(handle: Dpsr):
        import torch

        class _F(torch.autograd.Function):
            @staticmethod
            def forward(ctx, points, normals):
                chi = handle.forward(points.contiguous(), normals.contiguous())
                ctx.save_for_backward(points, normals, chi)
                ctx.epoch = handle.epoch
                return chi

            @staticmethod
            def backward(ctx, grad_chi):
                points, normals, chi = ctx.saved_tensors
                handle.check_epoch(ctx.epoch)   # a later forward on this handle has replaced the bins and statistics
                gp, gn = handle.backward(points.contiguous(), normals.contiguous(), chi, grad_chi.contiguous())
                return gp, gn

        return _F.apply


def dpsr(handle: Dpsr):
    return DpsrFunction.make(handle)

"""Thin Python binding of libhaccpm.so (include/haccpm.h): argument marshalling only.
The long-range particle-mesh force of PAPER.md section 2.3 runs in the library's CUDA kernels
and cuFFT; PyTorch provides device memory and the stream.  No CPU fallback."""
from __future__ import annotations

import ctypes as C

import torch

from . import build as _build

_lib = None
OK, EINVAL, ENOMEM, ECUDA, EDATA = 0, -1, -3, -4, -5

ABI_SYMBOLS = ("haccpm_abi_version", "haccpm_workspace_bytes", "haccpm_create", "haccpm_destroy",
               "hacc_lr_force", "haccpm_get_density", "haccpm_sync")


class HaccpmError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: status {status}")


def lib() -> C.CDLL:
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(_build.build_pm())
    vp, i64, f32 = C.c_void_p, C.c_int64, C.c_float
    L.haccpm_abi_version.restype = C.c_int
    L.haccpm_workspace_bytes.restype = C.c_size_t
    L.haccpm_workspace_bytes.argtypes = [C.c_int]
    L.haccpm_create.restype = C.c_int
    L.haccpm_create.argtypes = [C.POINTER(vp), C.c_int, f32, f32, C.c_int, vp, C.c_size_t, vp]
    L.haccpm_destroy.restype = C.c_int
    L.haccpm_destroy.argtypes = [vp]
    L.hacc_lr_force.restype = C.c_int
    L.hacc_lr_force.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp, f32, vp, vp, vp]
    L.haccpm_get_density.restype = C.c_int
    L.haccpm_get_density.argtypes = [vp, C.POINTER(vp)]
    L.haccpm_sync.restype = C.c_int
    L.haccpm_sync.argtypes = [vp]
    _lib = L
    return L


def _check(status, where):
    if status != OK:
        raise HaccpmError(status, where)


def _ptr(t, n, name):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float32 \
            or not t.is_contiguous() or t.numel() < n:
        raise TypeError(f"{name}: expected a contiguous float32 CUDA tensor of >= {n} elements")
    return C.c_void_p(t.data_ptr())


class Context:
    def __init__(self, ng: int, box_l: float, sigma: float = 0.8, n_s: int = 3, device="cuda:0",
                 stream=None):
        if not torch.cuda.is_available():
            raise HaccpmError(ECUDA, "haccpm_create (no CUDA device; there is no CPU path)")
        self.device = torch.device(device)
        self.ng, self.box_l = int(ng), float(box_l)
        nbytes = int(lib().haccpm_workspace_bytes(self.ng))
        if nbytes == 0:
            raise HaccpmError(EINVAL, "haccpm_workspace_bytes")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            self._ws_ptr = (self.workspace.data_ptr() + 255) & ~255
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            _check(lib().haccpm_create(C.byref(h), self.ng, self.box_l, float(sigma), int(n_s),
                                       C.c_void_p(self._ws_ptr), nbytes,
                                       C.c_void_p(self.stream.cuda_stream)), "haccpm_create")
        self.handle = h

    def close(self):
        if getattr(self, "handle", None):
            lib().haccpm_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def hacc_lr_force(ctx: Context, x, y, z, mass, ax, ay, az, dt=0.0, vx=None, vy=None, vz=None):
    n = x.numel()
    _check(lib().hacc_lr_force(ctx.handle, n, _ptr(x, n, "x"), _ptr(y, n, "y"), _ptr(z, n, "z"),
                               _ptr(mass, n, "mass"), _ptr(ax, n, "ax"), _ptr(ay, n, "ay"),
                               _ptr(az, n, "az"), float(dt), _ptr(vx, n, "vx"), _ptr(vy, n, "vy"),
                               _ptr(vz, n, "vz")), "hacc_lr_force")


def haccpm_get_density(ctx: Context):
    """A copy of the deposited density grid, shape (ng, ng, ng)."""
    p = C.c_void_p()
    _check(lib().haccpm_get_density(ctx.handle, C.byref(p)), "haccpm_get_density")
    haccpm_sync(ctx)
    off = p.value - ctx.workspace.data_ptr()
    ng = ctx.ng
    return ctx.workspace[off:off + 4 * ng ** 3].view(torch.float32).reshape(ng, ng, ng).clone()


def haccpm_sync(ctx: Context):
    _check(lib().haccpm_sync(ctx.handle), "haccpm_sync")

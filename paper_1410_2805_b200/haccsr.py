"""Thin Python binding of libhaccsr.so (include/haccsr.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch is used for device
memory (tensors -> data_ptr()) and the stream.  There is no CPU fallback: if the library is
missing it is built with nvcc, and if that fails the import raises.

Module-level functions carry the ABI's names (`hacc_sr_bin`, `hacc_sr_force`, `hacc_sr_kick`,
`hacc_sr_force_kick`, `hacc_sr_drift`, `haccsr_*`); `Context` owns the workspace tensor.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import torch

from . import build as _build

_lib = None

OK, EINVAL, ESTATE, ENOMEM, ECUDA, EDATA = 0, -1, -2, -3, -4, -5

ABI_SYMBOLS = (
    "haccsr_abi_version", "haccsr_workspace_bytes", "haccsr_create", "haccsr_destroy",
    "haccsr_workspace_bytes_slab", "haccsr_create_slab", "hacc_sr_pack_layer", "hacc_sr_unpack",
    "hacc_sr_bin", "hacc_sr_force", "hacc_sr_kick", "hacc_sr_force_kick", "hacc_sr_drift",
    "hacc_sr_subcycle", "hacc_sr_subcycle_multilevel",
    "haccsr_get_mesh", "haccsr_get_stats", "haccsr_sync", "haccsr_strerror",
    "haccsr_probe_peak", "hacc_sr_cell_start_noalloc",
)

NOALLOC_MAX_NC = 64   # HACCSR_NOALLOC_MAX_NC of include/haccsr.h


class HaccsrError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {strerror(status)} ({status})")


class _Stats(C.Structure):
    _fields_ = [("n", C.c_int64), ("n_cells", C.c_int64), ("n_eval", C.c_uint64),
                ("n_items", C.c_uint32), ("n_split_items", C.c_uint32),
                ("max_cell_count", C.c_uint32), ("sources_per_split", C.c_uint32),
                ("n_recheck_tiles", C.c_uint64)]


def lib() -> C.CDLL:
    """Load (building if needed) libhaccsr.so and declare the ABI's signatures."""
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(_build.build())
    vp, i64, f32, u64 = C.c_void_p, C.c_int64, C.c_float, C.c_uint64
    L.haccsr_abi_version.restype = C.c_int
    L.haccsr_abi_version.argtypes = []
    L.haccsr_workspace_bytes.restype = C.c_size_t
    L.haccsr_workspace_bytes.argtypes = [i64, C.c_int]
    L.haccsr_create.restype = C.c_int
    L.haccsr_create.argtypes = [C.POINTER(vp), i64, f32, C.c_int, vp, C.c_size_t, vp]
    L.haccsr_destroy.restype = C.c_int
    L.haccsr_destroy.argtypes = [vp]
    L.haccsr_workspace_bytes_slab.restype = C.c_size_t
    L.haccsr_workspace_bytes_slab.argtypes = [i64, C.c_int, C.c_int]
    L.haccsr_create_slab.restype = C.c_int
    L.haccsr_create_slab.argtypes = [C.POINTER(vp), i64, f32, C.c_int, C.c_int, C.c_int, vp,
                                     C.c_size_t, vp]
    L.hacc_sr_pack_layer.restype = C.c_int
    L.hacc_sr_pack_layer.argtypes = [vp, i64, vp, vp, vp, vp, C.c_int, vp, i64, vp]
    L.hacc_sr_unpack.restype = C.c_int
    L.hacc_sr_unpack.argtypes = [vp, i64, vp, vp, vp, vp, vp]
    L.hacc_sr_bin.restype = C.c_int
    L.hacc_sr_bin.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp]
    L.hacc_sr_force.restype = C.c_int
    L.hacc_sr_force.argtypes = [vp, f32, f32, C.POINTER(f32), vp, vp, vp, vp, vp]
    L.hacc_sr_kick.restype = C.c_int
    L.hacc_sr_kick.argtypes = [vp, f32]
    L.hacc_sr_force_kick.restype = C.c_int
    L.hacc_sr_force_kick.argtypes = [vp, f32, f32, C.POINTER(f32), f32, vp, vp, vp, vp, vp]
    L.hacc_sr_drift.restype = C.c_int
    L.hacc_sr_drift.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, f32]
    L.hacc_sr_subcycle.restype = C.c_int
    L.hacc_sr_subcycle.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp, f32, f32, C.POINTER(f32),
                                   f32, C.c_int, vp, vp, vp]
    L.hacc_sr_subcycle_multilevel.restype = C.c_int
    L.hacc_sr_subcycle_multilevel.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp, f32, f32,
                                              C.POINTER(f32), f32, f32, C.c_int, C.c_int, vp, vp,
                                              vp, vp, vp]
    L.haccsr_get_mesh.restype = C.c_int
    L.haccsr_get_mesh.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp),
                                  C.POINTER(vp)]
    L.haccsr_get_stats.restype = C.c_int
    L.haccsr_get_stats.argtypes = [vp, C.POINTER(_Stats)]
    L.haccsr_sync.restype = C.c_int
    L.haccsr_sync.argtypes = [vp]
    L.haccsr_strerror.restype = C.c_char_p
    L.haccsr_strerror.argtypes = [C.c_int]
    L.hacc_sr_cell_start_noalloc.restype = C.c_int
    L.hacc_sr_cell_start_noalloc.argtypes = [i64, vp, vp, vp, f32, C.c_int, vp, vp]
    L.haccsr_probe_peak.restype = C.c_int
    L.haccsr_probe_peak.argtypes = [C.c_int, C.c_int, vp, C.POINTER(C.c_double),
                                    C.POINTER(C.c_double)]
    _lib = L
    return L


def strerror(status: int) -> str:
    return lib().haccsr_strerror(int(status)).decode()


def _check(status: int, where: str):
    if status != OK:
        raise HaccsrError(status, where)


def _ptr(t, dtype, n=None, name="tensor"):
    """Device pointer of a contiguous CUDA tensor of the given dtype (None -> NULL)."""
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name}: expected a CUDA tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name}: expected contiguous {dtype}, got {t.dtype}")
    if n is not None and t.numel() < n:
        raise ValueError(f"{name}: needs {n} elements, has {t.numel()}")
    return C.c_void_p(t.data_ptr())


def _poly(poly):
    arr = (C.c_float * 6)(*[float(v) for v in poly])
    return arr


def haccsr_workspace_bytes(n_max: int, nc: int) -> int:
    return int(lib().haccsr_workspace_bytes(int(n_max), int(nc)))


@dataclass
class Stats:
    n: int
    n_cells: int
    n_eval: int
    n_items: int
    n_split_items: int
    max_cell_count: int
    sources_per_split: int
    n_recheck_tiles: int


class Context:
    """haccsr_ctx plus the torch workspace tensor that backs it."""

    def __init__(self, n_max: int, box_l: float, nc: int, device="cuda:0", stream=None,
                 slab=None):
        """slab=(cz_lo, nz_own): an overloaded slab context (haccsr_create_slab)."""
        if not torch.cuda.is_available():
            raise HaccsrError(ECUDA, "haccsr_create (no CUDA device; there is no CPU path)")
        self.device = torch.device(device)
        self.n_max, self.box_l, self.nc = int(n_max), float(box_l), int(nc)
        self.slab = None if slab is None else (int(slab[0]), int(slab[1]))
        self.nz = self.nc if slab is None else self.slab[1] + 2
        nbytes = (haccsr_workspace_bytes(n_max, nc) if slab is None else
                  int(lib().haccsr_workspace_bytes_slab(int(n_max), int(nc), self.slab[1])))
        if nbytes == 0:
            raise HaccsrError(EINVAL, "haccsr_workspace_bytes")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) & ~255
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            if slab is None:
                _check(lib().haccsr_create(C.byref(h), self.n_max, self.box_l, self.nc,
                                           C.c_void_p(self._ws_ptr), nbytes,
                                           C.c_void_p(self.stream.cuda_stream)), "haccsr_create")
            else:
                _check(lib().haccsr_create_slab(C.byref(h), self.n_max, self.box_l, self.nc,
                                                self.slab[0], self.slab[1],
                                                C.c_void_p(self._ws_ptr), nbytes,
                                                C.c_void_p(self.stream.cuda_stream)),
                       "haccsr_create_slab")
        self.handle = h
        self.n = 0
        self._keep = []  # tensors the C side holds pointers to

    def close(self):
        if getattr(self, "handle", None):
            lib().haccsr_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def haccsr_create(n_max, box_l, nc, device="cuda:0", stream=None) -> Context:
    return Context(n_max, box_l, nc, device, stream)


def haccsr_destroy(ctx: Context):
    ctx.close()


def hacc_sr_bin(ctx: Context, x, y, z, mass=None, vx=None, vy=None, vz=None):
    n = x.numel()
    f = torch.float32
    _check(lib().hacc_sr_bin(ctx.handle, n, _ptr(x, f, n, "x"), _ptr(y, f, n, "y"),
                             _ptr(z, f, n, "z"), _ptr(mass, f, n, "mass"),
                             _ptr(vx, f, n, "vx"), _ptr(vy, f, n, "vy"), _ptr(vz, f, n, "vz")),
           "hacc_sr_bin")
    ctx.n = n
    ctx._keep = [vx, vy, vz]


def hacc_sr_force(ctx: Context, eps, r_max, poly, ax, ay, az, nbr_count=None, pair_total=None):
    n, f = ctx.n, torch.float32
    _check(lib().hacc_sr_force(ctx.handle, float(eps), float(r_max), _poly(poly),
                               _ptr(ax, f, n, "ax"), _ptr(ay, f, n, "ay"), _ptr(az, f, n, "az"),
                               _ptr(nbr_count, torch.int32, n, "nbr_count"),
                               _ptr(pair_total, torch.int64, 1, "pair_total")),
           "hacc_sr_force")
    ctx._keep = ctx._keep[:3] + [ax, ay, az]


def hacc_sr_force_kick(ctx: Context, eps, r_max, poly, dt, ax, ay, az, nbr_count=None,
                       pair_total=None):
    n, f = ctx.n, torch.float32
    _check(lib().hacc_sr_force_kick(ctx.handle, float(eps), float(r_max), _poly(poly), float(dt),
                                    _ptr(ax, f, n, "ax"), _ptr(ay, f, n, "ay"),
                                    _ptr(az, f, n, "az"),
                                    _ptr(nbr_count, torch.int32, n, "nbr_count"),
                                    _ptr(pair_total, torch.int64, 1, "pair_total")),
           "hacc_sr_force_kick")
    ctx._keep = ctx._keep[:3] + [ax, ay, az]


def hacc_sr_kick(ctx: Context, dt):
    _check(lib().hacc_sr_kick(ctx.handle, float(dt)), "hacc_sr_kick")


def hacc_sr_drift(ctx: Context, x, y, z, vx, vy, vz, dt):
    n, f = x.numel(), torch.float32
    _check(lib().hacc_sr_drift(ctx.handle, n, _ptr(x, f, n, "x"), _ptr(y, f, n, "y"),
                               _ptr(z, f, n, "z"), _ptr(vx, f, n, "vx"), _ptr(vy, f, n, "vy"),
                               _ptr(vz, f, n, "vz"), float(dt)), "hacc_sr_drift")


def hacc_sr_subcycle(ctx: Context, x, y, z, mass, vx, vy, vz, eps, r_max, poly, dt, n_sub,
                     ax, ay, az):
    n, f = x.numel(), torch.float32
    _check(lib().hacc_sr_subcycle(ctx.handle, n, _ptr(x, f, n, "x"), _ptr(y, f, n, "y"),
                                  _ptr(z, f, n, "z"), _ptr(mass, f, n, "mass"),
                                  _ptr(vx, f, n, "vx"), _ptr(vy, f, n, "vy"),
                                  _ptr(vz, f, n, "vz"), float(eps), float(r_max), _poly(poly),
                                  float(dt), int(n_sub), _ptr(ax, f, n, "ax"),
                                  _ptr(ay, f, n, "ay"), _ptr(az, f, n, "az")),
           "hacc_sr_subcycle")
    ctx.n = n
    ctx._keep = [vx, vy, vz, ax, ay, az]


def hacc_sr_subcycle_multilevel(ctx: Context, x, y, z, mass, vx, vy, vz, eps, r_max, poly, T, d,
                                l_min, l_max, ax, ay, az, level, evals=None):
    """level: uint8 CUDA tensor (n); evals: int64 CUDA tensor (1) or None."""
    n, f = x.numel(), torch.float32
    _check(lib().hacc_sr_subcycle_multilevel(
        ctx.handle, n, _ptr(x, f, n, "x"), _ptr(y, f, n, "y"), _ptr(z, f, n, "z"),
        _ptr(mass, f, n, "mass"), _ptr(vx, f, n, "vx"), _ptr(vy, f, n, "vy"),
        _ptr(vz, f, n, "vz"), float(eps), float(r_max), _poly(poly), float(T), float(d),
        int(l_min), int(l_max), _ptr(ax, f, n, "ax"), _ptr(ay, f, n, "ay"), _ptr(az, f, n, "az"),
        _ptr(level, torch.uint8, n, "level"), _ptr(evals, torch.int64, 1, "evals")),
        "hacc_sr_subcycle_multilevel")
    ctx.n = n
    ctx._keep = [vx, vy, vz, ax, ay, az, level]


def haccsr_create_slab(n_max, box_l, nc, cz_lo, nz_own, device="cuda:0", stream=None) -> Context:
    return Context(n_max, box_l, nc, device, stream, slab=(cz_lo, nz_own))


def hacc_sr_pack_layer(ctx: Context, x, y, z, mass, cz_layer, out_records, count, n=None):
    """out_records: float32 CUDA tensor of 4*capacity elements; count: int32 tensor (1)."""
    n = x.numel() if n is None else int(n)
    f = torch.float32
    cap = out_records.numel() // 4
    _check(lib().hacc_sr_pack_layer(ctx.handle, n, _ptr(x, f, n, "x"), _ptr(y, f, n, "y"),
                                    _ptr(z, f, n, "z"), _ptr(mass, f, n, "mass"), int(cz_layer),
                                    _ptr(out_records, f, None, "out_records"), cap,
                                    _ptr(count, torch.int32, 1, "count")), "hacc_sr_pack_layer")


def hacc_sr_unpack(ctx: Context, records, n, x, y, z, mass=None):
    """Append n float4 records to the arrays x, y, z, (mass) -- pass views that start at the
    first free element."""
    f = torch.float32
    n = int(n)
    _check(lib().hacc_sr_unpack(ctx.handle, n, _ptr(records, f, 4 * n, "records"),
                                _ptr(x, f, n, "x"), _ptr(y, f, n, "y"), _ptr(z, f, n, "z"),
                                _ptr(mass, f, n, "mass")), "hacc_sr_unpack")


def haccsr_sync(ctx: Context):
    _check(lib().haccsr_sync(ctx.handle), "haccsr_sync")


def haccsr_get_stats(ctx: Context) -> Stats:
    s = _Stats()
    _check(lib().haccsr_get_stats(ctx.handle, C.byref(s)), "haccsr_get_stats")
    return Stats(*(int(getattr(s, k)) for k, _ in _Stats._fields_))


def haccsr_get_mesh(ctx: Context):
    """Copies of the mesh arrays as torch tensors: dict(cell_start, perm, sorted_pos, cell_id).

    uint32 arrays come back as int64 tensors (torch has no full uint32 support)."""
    ps = [C.c_void_p() for _ in range(4)]
    _check(lib().haccsr_get_mesh(ctx.handle, *[C.byref(p) for p in ps]), "haccsr_get_mesh")
    haccsr_sync(ctx)
    ws = ctx.workspace
    base = ws.data_ptr()

    def view(p, nbytes):
        off = p.value - base
        return ws[off:off + nbytes]

    n, cells = ctx.n, ctx.nc * ctx.nc * ctx.nz
    u32 = lambda p, k: view(p, 4 * k).view(torch.int32).to(torch.int64) & 0xFFFFFFFF
    return dict(cell_start=u32(ps[0], cells + 1), perm=u32(ps[1], n),
                sorted_pos=view(ps[2], 16 * n).view(torch.float32).reshape(n, 4).clone(),
                cell_id=u32(ps[3], n))


def haccsr_probe_peak(kind: int, reps: int = 3, stream=None):
    """(milliseconds, operations) of one peak-probe kernel; see include/haccsr.h."""
    ms, ops = C.c_double(), C.c_double()
    st = stream if stream is not None else torch.cuda.current_stream()
    _check(lib().haccsr_probe_peak(int(kind), int(reps), C.c_void_p(st.cuda_stream),
                                   C.byref(ms), C.byref(ops)), "haccsr_probe_peak")
    return ms.value, ops.value


def hacc_sr_cell_start_noalloc(x, y, z, box_l: float, nc: int, cell_start, stream=None):
    """cell_start[nc^3+1] of the chaining mesh with no context and no allocation in the library
    (its counters sit in a static device array: nc <= 64; see include/haccsr.h).

    `cell_start` is the caller's int32 CUDA tensor of at least nc^3+1 elements (the library
    writes uint32; torch has no full uint32 support).  Runs on x's device; calls that overlap on
    the GPU race on the shared array."""
    n = int(x.numel())
    if int(nc) > NOALLOC_MAX_NC:
        raise HaccsrError(ENOMEM, f"hacc_sr_cell_start_noalloc (nc = {int(nc)} > {NOALLOC_MAX_NC}:"
                                  " the mesh does not fit the library's static scratch array)")
    cells = int(nc) ** 3
    with torch.cuda.device(x.device):
        st = stream if stream is not None else torch.cuda.current_stream(x.device)
        _check(lib().hacc_sr_cell_start_noalloc(
            n, _ptr(x, torch.float32, n, "x"), _ptr(y, torch.float32, n, "y"),
            _ptr(z, torch.float32, n, "z"), float(box_l), int(nc),
            _ptr(cell_start, torch.int32, cells + 1, "cell_start"),
            C.c_void_p(st.cuda_stream)), "hacc_sr_cell_start_noalloc")
    return cell_start

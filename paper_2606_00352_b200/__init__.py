"""paper_2606_00352_b200 -- B200-native HiGS forward render path (arxiv/paper_2606_00352).

Thin ctypes binding over ``libhigs.so`` (C ABI declared in ``include/higs.h``): argument
marshalling only, every step of the frame runs in the library's sm_100a kernels.  PyTorch is used
for device memory and streams, nothing else.  There is no CPU fallback: if the library cannot be
loaded or no CUDA device is present, calls raise.

Module-level functions carry the C names (``higs_create``, ``higs_render``, ...); ``Renderer`` is
a small convenience wrapper holding a context.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path
from typing import Optional

import numpy as np

from . import build as _build

HIGS_OK, HIGS_E_ARG, HIGS_E_CUDA, HIGS_E_CAPACITY, HIGS_E_NOMEM = 0, -1, -2, -3, -4
HIGS_FLAG_STAGE_TIMERS, HIGS_FLAG_COUNT_EVALS, HIGS_FLAG_NO_XBATCH_CUT, HIGS_FLAG_RADIX_SORT, HIGS_FLAG_FP16, HIGS_FLAG_SH32 = 1, 2, 4, 8, 16, 32
HIGS_TILE, HIGS_MT_W, HIGS_MT_H, HIGS_MT_TILES, HIGS_BATCH_CAP = 8, 64, 32, 32, 1024

EXPORTS = ["higs_abi_version", "higs_strerror", "higs_last_error", "higs_create", "higs_destroy", "higs_set_flags",
           "higs_set_batch_cap", "higs_set_tile", "higs_set_macro_tile", "higs_sh32_encode_static", "higs_sh32_encode_static_error", "higs_render", "higs_render_host", "higs_scene_upload", "higs_render_view_host",
           "higs_render_view", "higs_scene_sort_spatial", "higs_scene_compress_sh", "higs_get_sh32", "higs_get_stats", "higs_get_lists", "higs_get_records", "higs_sort_segments", "higs_download"]


class higs_camera(C.Structure):
    _fields_ = [("view", C.c_float * 12), ("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float), ("cy", C.c_float),
                ("near_z", C.c_float), ("cam_pos", C.c_float * 3)]


class higs_stats(C.Structure):
    _fields_ = [("n_gaussians", C.c_int64), ("n_visible", C.c_int64), ("n_pairs", C.c_int64), ("n_units", C.c_int64),
                ("max_segment", C.c_int64), ("n_oversize", C.c_int64), ("n_mt_x", C.c_int32), ("n_mt_y", C.c_int32),
                ("batch_cap", C.c_int32), ("overflow", C.c_int32), ("n_launches", C.c_int32), ("tile", C.c_int32), ("n_evals", C.c_int64), ("n_tile_pairs", C.c_int64),
                ("ms_project", C.c_float), ("ms_count", C.c_float), ("ms_scan", C.c_float), ("ms_fill", C.c_float),
                ("ms_sort", C.c_float), ("ms_raster", C.c_float), ("ms_merge", C.c_float), ("ms_total", C.c_float)]

    def as_dict(self) -> dict:
        return {k: getattr(self, k) for k, _ in self._fields_}


class higs_lists(C.Structure):
    _fields_ = [("n_pairs", C.c_int64), ("n_units", C.c_int64), ("n_mt", C.c_int32), ("mt_count", C.c_void_p),
                ("mt_offset", C.c_void_p), ("batch_offset", C.c_void_p), ("pairs", C.c_void_p), ("unit_active", C.c_void_p), ("tile_load", C.c_void_p)]


class higs_records(C.Structure):
    _fields_ = [("n", C.c_int64), ("valid_bits", C.c_void_p), ("rec", C.c_void_p)]


class HigsError(RuntimeError):
    def __init__(self, status: int, what: str):
        super().__init__(f"{what}: status {status}")
        self.status = status


_lib = None


def lib_path() -> Path:
    return _build.LIB


def load() -> C.CDLL:
    """Load libhigs.so, building it first if it is missing or stale.  Raises if that fails."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(str(path))
        vp, f32p = C.c_void_p, C.c_void_p
        L.higs_abi_version.restype = C.c_int
        L.higs_strerror.restype = C.c_char_p; L.higs_strerror.argtypes = [C.c_int]
        L.higs_last_error.restype = C.c_char_p; L.higs_last_error.argtypes = [vp]
        L.higs_create.restype = C.c_int
        L.higs_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int64, C.c_int, C.c_int, C.c_int64]
        L.higs_destroy.restype = None; L.higs_destroy.argtypes = [vp]
        L.higs_set_flags.restype = C.c_int; L.higs_set_flags.argtypes = [vp, C.c_uint32]
        L.higs_set_batch_cap.restype = C.c_int; L.higs_set_batch_cap.argtypes = [vp, C.c_int]
        L.higs_set_tile.restype = C.c_int; L.higs_set_tile.argtypes = [vp, C.c_int]
        L.higs_set_macro_tile.restype = C.c_int; L.higs_set_macro_tile.argtypes = [vp, C.c_int, C.c_int]
        L.higs_sh32_encode_static.restype = C.c_int
        L.higs_sh32_encode_static.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.higs_sh32_encode_static_error.restype = C.c_char_p; L.higs_sh32_encode_static_error.argtypes = []
        L.higs_render.restype = C.c_int
        L.higs_render.argtypes = [vp, f32p, f32p, f32p, f32p, f32p, C.c_int, C.c_int64, C.POINTER(higs_camera),
                                  C.c_int, C.c_int, f32p, vp]
        L.higs_render_host.restype = C.c_int
        L.higs_render_host.argtypes = [vp, f32p, f32p, f32p, f32p, f32p, C.c_int, C.c_int64, C.POINTER(higs_camera),
                                       C.c_int, C.c_int, f32p]
        L.higs_scene_upload.restype = C.c_int
        L.higs_scene_upload.argtypes = [vp, f32p, f32p, f32p, f32p, f32p, C.c_int, C.c_int64]
        L.higs_render_view_host.restype = C.c_int
        L.higs_render_view_host.argtypes = [vp, C.POINTER(higs_camera), C.c_int, C.c_int, f32p]
        L.higs_render_view.restype = C.c_int
        L.higs_render_view.argtypes = [vp, C.POINTER(higs_camera), C.c_int, C.c_int, f32p, vp]
        L.higs_scene_sort_spatial.restype = C.c_int; L.higs_scene_sort_spatial.argtypes = [vp, vp]
        L.higs_scene_compress_sh.restype = C.c_int; L.higs_scene_compress_sh.argtypes = [vp]
        L.higs_get_sh32.restype = C.c_int; L.higs_get_sh32.argtypes = [vp, vp, vp]
        L.higs_get_stats.restype = C.c_int; L.higs_get_stats.argtypes = [vp, C.POINTER(higs_stats)]
        L.higs_get_lists.restype = C.c_int; L.higs_get_lists.argtypes = [vp, C.POINTER(higs_lists)]
        L.higs_get_records.restype = C.c_int; L.higs_get_records.argtypes = [vp, C.POINTER(higs_records)]
        L.higs_download.restype = C.c_int; L.higs_download.argtypes = [vp, vp, vp, C.c_uint64]
        L.higs_sort_segments.restype = C.c_int; L.higs_sort_segments.argtypes = [vp, vp, vp, C.c_int32, vp]
        _lib = L
    return _lib


def make_camera(cam) -> higs_camera:
    """higs_camera from anything with .as_floats() -> 20 floats (view[12], fx, fy, cx, cy, near_z, cam_pos[3])."""
    f = np.asarray(cam.as_floats() if hasattr(cam, "as_floats") else cam, dtype=np.float32)
    assert f.shape == (20,)
    c = higs_camera()
    C.memmove(C.byref(c), f.ctypes.data, 80)
    return c


def _ptr(t) -> Optional[int]:
    """Raw address of a torch tensor (device or host) or numpy array; checks fp32 + contiguity."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.dtype == np.float32 and t.flags["C_CONTIGUOUS"]
        return t.ctypes.data
    import torch
    assert t.dtype == torch.float32 and t.is_contiguous()
    return t.data_ptr()


def _check(status: int, what: str, ctx=None):
    if status != HIGS_OK:
        L = load()
        msg = L.higs_strerror(status).decode()
        if status == HIGS_E_CUDA and ctx:
            msg += ": " + L.higs_last_error(ctx).decode()
        raise HigsError(status, f"{what}: {msg}")


# ---- C-named functions ---------------------------------------------------------------------------
def higs_abi_version() -> int:
    return int(load().higs_abi_version())


def higs_create(device: int, max_gaussians: int, max_W: int, max_H: int, max_pairs: int = 0) -> C.c_void_p:
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2606_00352_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
    ctx = C.c_void_p()
    _check(load().higs_create(C.byref(ctx), device, max_gaussians, max_W, max_H, max_pairs), "higs_create")
    return ctx


def higs_destroy(ctx) -> None:
    load().higs_destroy(ctx)


def higs_set_flags(ctx, flags: int) -> None:
    _check(load().higs_set_flags(ctx, flags), "higs_set_flags", ctx)


def higs_set_batch_cap(ctx, batch_cap: int) -> None:
    _check(load().higs_set_batch_cap(ctx, batch_cap), "higs_set_batch_cap", ctx)


def higs_set_tile(ctx, tile: int) -> None:
    _check(load().higs_set_tile(ctx, tile), "higs_set_tile", ctx)


def higs_set_macro_tile(ctx, tiles_x: int, tiles_y: int) -> None:
    _check(load().higs_set_macro_tile(ctx, tiles_x, tiles_y), "higs_set_macro_tile", ctx)


def higs_render(ctx, means, scales, quats, opacities, sh, degree: int, cam: higs_camera, W: int, H: int, out_rgb,
                stream: Optional[int] = None) -> None:
    """Device tensors in, device tensor out; enqueues on `stream` (default: torch's current stream)."""
    import torch
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    N = int(opacities.shape[0])
    _check(load().higs_render(ctx, _ptr(means), _ptr(scales), _ptr(quats), _ptr(opacities), _ptr(sh), degree, N,
                              C.byref(cam), W, H, _ptr(out_rgb), C.c_void_p(stream)), "higs_render", ctx)


def higs_render_host(ctx, means, scales, quats, opacities, sh, degree: int, cam: higs_camera, W: int, H: int, out_rgb) -> None:
    """Host (numpy / CPU torch) buffers in and out; uploads, renders, downloads, synchronises."""
    N = int(opacities.shape[0])
    _check(load().higs_render_host(ctx, _ptr(means), _ptr(scales), _ptr(quats), _ptr(opacities), _ptr(sh), degree, N,
                                   C.byref(cam), W, H, _ptr(out_rgb)), "higs_render_host", ctx)


def higs_scene_upload(ctx, means, scales, quats, opacities, sh, degree: int) -> None:
    N = int(opacities.shape[0])
    _check(load().higs_scene_upload(ctx, _ptr(means), _ptr(scales), _ptr(quats), _ptr(opacities), _ptr(sh), degree, N),
           "higs_scene_upload", ctx)


def higs_scene_sort_spatial(ctx, n: int) -> np.ndarray:
    """Reorders the resident scene along a Morton curve; returns perm (uint32 [n]): new index i holds uploaded gaussian perm[i]."""
    perm = np.zeros(n, np.uint32)
    _check(load().higs_scene_sort_spatial(ctx, C.c_void_p(perm.ctypes.data)), "higs_scene_sort_spatial", ctx)
    return perm


def higs_scene_compress_sh(ctx) -> None:
    _check(load().higs_scene_compress_sh(ctx), "higs_scene_compress_sh", ctx)


def higs_get_sh32(ctx, n: int):
    """(codes [n][32] uint8, scales [16][3] float32) of the resident scene's 32-byte SH codes."""
    codes = np.zeros((n, 32), np.uint8); scales = np.zeros((16, 3), np.float32)
    _check(load().higs_get_sh32(ctx, C.c_void_p(codes.ctypes.data), C.c_void_p(scales.ctypes.data)), "higs_get_sh32", ctx)
    return codes, scales


HIGS_SH32_STATIC_MAX_N = 1 << 30


def higs_sh32_encode_static(d_sh, n: int, d_codes, d_scales, stream: Optional[int] = None) -> None:
    """32-byte SH codes of n degree-3 rows without any allocation (include/higs.h): device tensors in and out, enqueue only."""
    import torch
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    L = load()
    rc = L.higs_sh32_encode_static(C.c_void_p(d_sh.data_ptr() if d_sh is not None else None), int(n),
                                   C.c_void_p(d_codes.data_ptr() if d_codes is not None else None),
                                   C.c_void_p(d_scales.data_ptr() if d_scales is not None else None), C.c_void_p(stream))
    if rc != HIGS_OK:
        raise HigsError(rc, "higs_sh32_encode_static: " + L.higs_sh32_encode_static_error().decode())


def higs_render_view_host(ctx, cam: higs_camera, W: int, H: int, out_rgb) -> None:
    _check(load().higs_render_view_host(ctx, C.byref(cam), W, H, _ptr(out_rgb)), "higs_render_view_host", ctx)


def higs_render_view(ctx, cam: higs_camera, W: int, H: int, out_rgb, stream: Optional[int] = None) -> None:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    _check(load().higs_render_view(ctx, C.byref(cam), W, H, _ptr(out_rgb), C.c_void_p(stream)), "higs_render_view", ctx)


def higs_get_stats(ctx, allow_overflow: bool = False) -> dict:
    st = higs_stats()
    rc = load().higs_get_stats(ctx, C.byref(st))
    if not (allow_overflow and rc == HIGS_E_CAPACITY):
        _check(rc, "higs_get_stats", ctx)
    return st.as_dict()


def _dev_to_numpy(ctx, ptr, count: int, dtype) -> np.ndarray:
    """Copy `count` items of `dtype` from a device pointer of the context into numpy (higs_download)."""
    out = np.empty(count, dtype=np.dtype(dtype))
    if count:
        _check(load().higs_download(ctx, C.c_void_p(ptr), C.c_void_p(out.ctypes.data), out.nbytes), "higs_download", ctx)
    return out


def higs_get_lists(ctx) -> dict:
    """The integer lists of the last frame copied to numpy: mt_count, mt_offset, batch_offset, keys, ids, unit_active."""
    ls = higs_lists()
    _check(load().higs_get_lists(ctx, C.byref(ls)), "higs_get_lists", ctx)
    nm, npairs, nun = int(ls.n_mt), int(ls.n_pairs), int(ls.n_units)
    pairs = _dev_to_numpy(ctx, ls.pairs, npairs, np.uint64)
    return {"n_pairs": npairs, "n_units": nun, "n_mt": nm,
            "mt_count": _dev_to_numpy(ctx, ls.mt_count, nm, np.uint32),
            "mt_offset": _dev_to_numpy(ctx, ls.mt_offset, nm + 1, np.uint32),
            "batch_offset": _dev_to_numpy(ctx, ls.batch_offset, nm + 1, np.uint32),
            "keys": (pairs >> np.uint64(32)).astype(np.uint32), "ids": (pairs & np.uint64(0xffffffff)).astype(np.uint32),
            "unit_active": _dev_to_numpy(ctx, ls.unit_active, nun, np.uint32),
            "tile_load": _dev_to_numpy(ctx, ls.tile_load, nm * HIGS_MT_TILES, np.uint32).reshape(nm, HIGS_MT_TILES)}


def higs_get_records(ctx) -> dict:
    """Per-gaussian records of the last frame: valid (N,) bool, rec (N,16) (rows of culled gaussians are stale)."""
    rc_ = higs_records()
    _check(load().higs_get_records(ctx, C.byref(rc_)), "higs_get_records", ctx)
    n = int(rc_.n)
    words = _dev_to_numpy(ctx, rc_.valid_bits, (n + 31) // 32, np.uint32)
    valid = ((words[:, None] >> np.arange(32, dtype=np.uint32)[None, :]) & 1).astype(bool).reshape(-1)[:n]
    return {"n": n, "valid": valid, "rec": _dev_to_numpy(ctx, rc_.rec, n * 16, np.float32).reshape(n, 16)}


def higs_sort_segments(ctx, pairs, seg_offset, stream: Optional[int] = None) -> None:
    """In-place segmented sort of a device int64/uint64 tensor `pairs`; seg_offset: device int32 tensor [n_seg+1]."""
    import torch
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    assert pairs.is_cuda and seg_offset.is_cuda and pairs.element_size() == 8 and seg_offset.element_size() == 4
    _check(load().higs_sort_segments(ctx, C.c_void_p(pairs.data_ptr()), C.c_void_p(seg_offset.data_ptr()),
                                     int(seg_offset.numel()) - 1, C.c_void_p(stream)), "higs_sort_segments", ctx)


# ---- convenience wrapper ------------------------------------------------------------------------
class Renderer:
    """Owns a higs_ctx.  render(scene tensors on the device, camera) -> (H, W, 3) fp32 device tensor."""

    def __init__(self, max_gaussians: int, max_W: int, max_H: int, max_pairs: int = 0, device: int = 0,
                 flags: int = 0, batch_cap: int = HIGS_BATCH_CAP, tile: int = HIGS_TILE, mt: tuple = (8, 4)):
        self.ctx = higs_create(device, max_gaussians, max_W, max_H, max_pairs)
        self.device = device
        if tile != HIGS_TILE:
            higs_set_tile(self.ctx, tile)
        if tuple(mt) != (8, 4):
            higs_set_macro_tile(self.ctx, int(mt[0]), int(mt[1]))
        if flags:
            higs_set_flags(self.ctx, flags)
        if batch_cap != HIGS_BATCH_CAP:
            higs_set_batch_cap(self.ctx, batch_cap)

    def close(self):
        if self.ctx is not None:
            higs_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def render(self, means, scales, quats, opacities, sh, degree, cam, out=None):
        import torch
        W, H = int(cam.W), int(cam.H)
        if out is None:
            out = torch.empty((H, W, 3), dtype=torch.float32, device=means.device)
        higs_render(self.ctx, means, scales, quats, opacities, sh, degree, make_camera(cam), W, H, out)
        return out

    def stats(self, allow_overflow: bool = False) -> dict:
        return higs_get_stats(self.ctx, allow_overflow)

    def lists(self) -> dict:
        return higs_get_lists(self.ctx)

    def records(self) -> dict:
        return higs_get_records(self.ctx)


def scene_to_device(scene, device: str = "cuda:0"):
    """Upload a higs_scenes.Scene's arrays as contiguous fp32 device tensors."""
    import torch
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(device)
    return f(scene.means), f(scene.scales), f(scene.quats), f(scene.opacities), f(scene.sh)

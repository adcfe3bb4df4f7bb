"""ctypes front-end of the CPU oracle (``higs_oracle.c``).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.  It
imports nothing from ``paper_2606_00352_b200`` and shares no code with it; the only module
both sides use is ``higs_scenes`` (seeded input generators, no method arithmetic).

See the header of ``higs_oracle.c`` for what each routine computes and which passage of the
paper it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from pathlib import Path
from typing import Optional, Tuple

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "higs_oracle.c"
_LIB = _HERE / "libhigs_oracle.so"

# -ffp-contract=off / -fno-fast-math are REQUIRED: the decision arithmetic is one rounding per
# written op.  -mfma only lets fmaf() compile to a hardware fma (the result is the same).
CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math", "-mfma",
          "-Wall", "-Wextra", "-pthread"]

MT_W, MT_H, TILE = 64, 32, 8
B_R = 1024


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (seconds).  Rebuilds when the source is newer."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", *CFLAGS, "-o", str(_LIB), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        f32p, f64p = C.POINTER(C.c_float), C.POINTER(C.c_double)
        u8p, u32p, i32p = C.POINTER(C.c_uint8), C.POINTER(C.c_uint32), C.POINTER(C.c_int32)
        L.orc_ln_spec.restype = C.c_float
        L.orc_ln_spec.argtypes = [C.c_float]
        L.orc_sh_basis.restype = None
        L.orc_sh_basis.argtypes = [f64p, f64p]
        L.orc_project.restype = C.c_int64
        L.orc_project.argtypes = [C.c_int64, f32p, f32p, f32p, f32p, f32p, C.c_int, f32p, C.c_int, C.c_int,
                                  u8p, u8p, u32p, f32p, f32p, f64p]
        L.orc_project_f64.restype = None
        L.orc_project_f64.argtypes = [f32p, f32p, f32p, C.c_float, f32p, C.c_int, C.c_int, f64p, f64p]
        L.orc_scan.restype = C.c_int
        L.orc_scan.argtypes = [f32p, C.c_int, C.c_int, C.c_int, C.c_int, i32p, C.c_int]
        L.orc_bin.restype = C.c_int64
        L.orc_bin.argtypes = [C.c_int64, u8p, u32p, f32p, C.c_int, C.c_int, C.c_int, u32p, u32p, u32p,
                              u32p, u32p, C.c_int64]
        L.orc_pixel_q.restype = C.c_float
        L.orc_pixel_q.argtypes = [C.c_float] * 7
        for name in ("orc_render", "orc_brute"):
            fn = getattr(L, name)
            fn.restype = C.c_int64
            fn.argtypes = [C.c_int64, u8p, u32p, f32p, f32p, f32p, f64p, C.c_int, C.c_int, C.c_int, C.c_int,
                           C.c_int, C.c_int, f64p, f64p]
        L.orc_bin_tile.restype = C.c_int64
        L.orc_bin_tile.argtypes = [C.c_int64, u8p, u32p, f32p, C.c_int, C.c_int, C.c_int, C.c_int, u32p, u32p, u32p, u32p, u32p, C.c_int64]
        L.orc_render_batched_tile.restype = None
        L.orc_render_batched_tile.argtypes = [u32p, u32p, f32p, f32p, f32p, f64p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, f64p]
        L.orc_bin_grid.restype = C.c_int64
        L.orc_bin_grid.argtypes = [C.c_int64, u8p, u32p, f32p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, u32p, u32p, u32p, u32p, u32p, C.c_int64]
        L.orc_render_batched_grid.restype = None
        L.orc_render_batched_grid.argtypes = [u32p, u32p, f32p, f32p, f32p, f64p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, f64p]
        L.orc_sh32_scales.restype = None; L.orc_sh32_scales.argtypes = [C.c_int64, f32p, f32p]
        L.orc_sh32_encode.restype = None; L.orc_sh32_encode.argtypes = [C.c_int64, f32p, f32p, u8p]
        L.orc_sh32_decode.restype = None; L.orc_sh32_decode.argtypes = [C.c_int64, u8p, f32p, f32p]
        L.orc_cholesky.restype = None
        L.orc_cholesky.argtypes = [C.c_double, C.c_double, C.c_double, f64p]
        L.orc_q_cholesky.restype = C.c_double
        L.orc_q_cholesky.argtypes = [C.c_double, C.c_double, f64p]
        L.orc_render_batched.restype = None
        L.orc_render_batched.argtypes = [u32p, u32p, f32p, f32p, f32p, f64p, C.c_int, C.c_int, C.c_int, C.c_int, f64p]
        _lib = L
    return _lib


def _p(a: Optional[np.ndarray], ctype):
    if a is None:
        return None
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(ctype))


def n_threads() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:  # pragma: no cover
        return max(1, os.cpu_count() or 1)


@dataclass
class Projected:
    """Per-gaussian records (O-LIST step 1)."""
    N: int
    W: int
    H: int
    n_vis: int
    valid: np.ndarray    # (N,) uint8
    reason: np.ndarray   # (N,) uint8 cull reason (0 = kept)
    key: np.ndarray      # (N,) uint32 depth key = bits(z_cam)
    geo: np.ndarray      # (N,9) float32: mux, muy, a, b, c, tau, hx, hy, tau_s (scan / bbox threshold)
    conic: np.ndarray    # (N,3) float32: A, B2, C
    rgb: np.ndarray      # (N,3) float64
    opac: np.ndarray     # (N,) float32 (input opacities)


@dataclass
class Lists:
    """O-LIST steps 2-5."""
    n_pairs: int
    n_units: int
    mt_count: np.ndarray      # (N_M,) uint32
    mt_offset: np.ndarray     # (N_M+1,) uint32
    batch_offset: np.ndarray  # (N_M+1,) uint32
    keys: np.ndarray          # (n_pairs,) uint32
    ids: np.ndarray           # (n_pairs,) uint32


def grid_dims(W: int, H: int) -> Tuple[int, int]:
    return (W + MT_W - 1) // MT_W, (H + MT_H - 1) // MT_H


def ln_spec(x: float) -> float:
    return float(lib().orc_ln_spec(C.c_float(x)))


def sh_basis(d) -> np.ndarray:
    d = np.ascontiguousarray(d, dtype=np.float64)
    Y = np.zeros(16, dtype=np.float64)
    lib().orc_sh_basis(_p(d, C.c_double), _p(Y, C.c_double))
    return Y


def pixel_q(px, py, mux, muy, A, B2, Cc) -> float:
    return float(lib().orc_pixel_q(*(C.c_float(v) for v in (px, py, mux, muy, A, B2, Cc))))


def project(scene, cam) -> Projected:
    N = scene.N
    means = np.ascontiguousarray(scene.means, dtype=np.float32)
    scales = np.ascontiguousarray(scene.scales, dtype=np.float32)
    quats = np.ascontiguousarray(scene.quats, dtype=np.float32)
    opac = np.ascontiguousarray(scene.opacities, dtype=np.float32)
    sh = np.ascontiguousarray(scene.sh, dtype=np.float32)
    camf = cam.as_floats()
    valid = np.zeros(N, np.uint8); reason = np.zeros(N, np.uint8); key = np.zeros(N, np.uint32)
    geo = np.zeros((N, 9), np.float32); conic = np.zeros((N, 3), np.float32); rgb = np.zeros((N, 3), np.float64)
    nvis = lib().orc_project(N, _p(means, C.c_float), _p(scales, C.c_float), _p(quats, C.c_float),
                             _p(opac, C.c_float), _p(sh, C.c_float), scene.degree, _p(camf, C.c_float),
                             cam.W, cam.H, _p(valid, C.c_uint8), _p(reason, C.c_uint8), _p(key, C.c_uint32),
                             _p(geo, C.c_float), _p(conic, C.c_float), _p(rgb, C.c_double))
    return Projected(N, cam.W, cam.H, int(nvis), valid, reason, key, geo, conic, rgb, opac)


def project_f64(mean, scale, quat, opacity, cam):
    """Plain fp64 definition of the projection of ONE gaussian: dict of mux, muy, a, b, c, A, B2, C, tau, zc."""
    m = np.ascontiguousarray(mean, np.float32); s = np.ascontiguousarray(scale, np.float32)
    q = np.ascontiguousarray(quat, np.float32); camf = cam.as_floats()
    out = np.zeros(9, np.float64); zc = np.zeros(1, np.float64)
    lib().orc_project_f64(_p(m, C.c_float), _p(s, C.c_float), _p(q, C.c_float), C.c_float(float(opacity)),
                          _p(camf, C.c_float), cam.W, cam.H, _p(out, C.c_double), _p(zc, C.c_double))
    names = ["mux", "muy", "a", "b", "c", "A", "B2", "C", "tau"]
    d = {k: float(v) for k, v in zip(names, out)}
    d["zc"] = float(zc[0])
    return d


def scan(geo_row: np.ndarray, W: int, H: int, cw: int = MT_W, ch: int = MT_H) -> np.ndarray:
    """Cell ids (r*ncx + m) the threshold ellipse of one gaussian touches (N-SCAN)."""
    g = np.ascontiguousarray(geo_row, np.float32)
    ncx, ncy = (W + cw - 1) // cw, (H + ch - 1) // ch
    out = np.zeros(ncx * ncy, np.int32)
    n = lib().orc_scan(_p(g, C.c_float), W, H, cw, ch, _p(out, C.c_int32), out.size)
    return out[:n].copy()


def bin_lists(pr: Projected, B_r: int = B_R, tile: int = TILE, mt: tuple = (8, 4)) -> Lists:
    """O-LIST.  tile = render-tile edge (8, or 16 for the variant of PAPER.md:286-299); mt = render tiles per macro-tile
    in x and y (the paper's 8 x 4; 4 x 8 and 16 x 2 for the shape sweep)."""
    mw, mh = mt[0] * tile, mt[1] * tile
    nmx, nmy = (pr.W + mw - 1) // mw, (pr.H + mh - 1) // mh
    NM = nmx * nmy
    mt_count = np.zeros(NM, np.uint32); mt_offset = np.zeros(NM + 1, np.uint32); batch_offset = np.zeros(NM + 1, np.uint32)
    args = (pr.N, _p(pr.valid, C.c_uint8), _p(pr.key, C.c_uint32), _p(pr.geo, C.c_float), pr.W, pr.H, B_r, mw, mh,
            _p(mt_count, C.c_uint32), _p(mt_offset, C.c_uint32), _p(batch_offset, C.c_uint32))
    npairs = int(lib().orc_bin_grid(*args, None, None, 0))
    keys = np.zeros(max(npairs, 1), np.uint32); ids = np.zeros(max(npairs, 1), np.uint32)
    lib().orc_bin_grid(*args, _p(keys, C.c_uint32), _p(ids, C.c_uint32), npairs)
    return Lists(npairs, int(batch_offset[NM]), mt_count, mt_offset, batch_offset, keys[:npairs], ids[:npairs])


def _render(fn, pr: Projected, window, terminate, threads, want_T):
    x0, y0, x1, y1 = window if window is not None else (0, 0, pr.W, pr.H)
    ww, hh = x1 - x0, y1 - y0
    out = np.zeros((hh, ww, 3), np.float64)
    outT = np.zeros((hh, ww), np.float64)
    n = fn(pr.N, _p(pr.valid, C.c_uint8), _p(pr.key, C.c_uint32), _p(pr.geo, C.c_float), _p(pr.conic, C.c_float),
           _p(pr.opac, C.c_float), _p(pr.rgb, C.c_double), x0, y0, x1, y1, int(terminate),
           int(threads or n_threads()), _p(out, C.c_double), _p(outT, C.c_double))
    return (out, outT, int(n)) if want_T else out


def render(pr: Projected, window=None, terminate: bool = True, threads: Optional[int] = None, want_T: bool = False):
    """O-IMG, gaussian-major untiled renderer.  window = (x0, y0, x1, y1) or None for the full image."""
    return _render(lib().orc_render, pr, window, terminate, threads, want_T)


def brute(pr: Projected, window=None, terminate: bool = True, threads: Optional[int] = None, want_T: bool = False):
    """O-IMG with no bounding box: every pixel tests every valid gaussian (tiny scenes only)."""
    return _render(lib().orc_brute, pr, window, terminate, threads, want_T)


def render_batched(pr: Projected, ls: Lists, B_r: int = B_R, terminate: bool = True, tile: int = TILE, mt: tuple = (8, 4)) -> np.ndarray:
    """The method step by step: per-macro-tile lists, batches of B_r, Eq. (1) merge."""
    out = np.zeros((pr.H, pr.W, 3), np.float64)
    ids = ls.ids if ls.ids.size else np.zeros(1, np.uint32)
    lib().orc_render_batched_grid(_p(ls.mt_offset, C.c_uint32), _p(ids, C.c_uint32), _p(pr.geo, C.c_float),
                                  _p(pr.conic, C.c_float), _p(pr.opac, C.c_float), _p(pr.rgb, C.c_double),
                                  pr.W, pr.H, B_r, mt[0] * tile, mt[1] * tile, int(terminate), _p(out, C.c_double))
    return out


def cholesky(a: float, b: float, c: float) -> np.ndarray:
    """(l0, l1, l2) with Sigma^-1 = L L^T, L = [[l0, 0], [l1, l2]], from the 2D covariance, fp64."""
    l = np.zeros(3, np.float64)
    lib().orc_cholesky(float(a), float(b), float(c), _p(l, C.c_double))
    return l


def q_cholesky(dx: float, dy: float, l: np.ndarray) -> float:
    """q = (l0 dx + l1 dy)^2 + (l2 dy)^2, fp64."""
    return float(lib().orc_q_cholesky(float(dx), float(dy), _p(np.ascontiguousarray(l, np.float64), C.c_double)))


def render_scene(scene, cam, window=None, threads: Optional[int] = None) -> np.ndarray:
    """project -> O-IMG; what bench.py's cpu_baseline leg times."""
    return render(project(scene, cam), window=window, threads=threads)


# ---- 32-byte SH codec (layout: DESIGN.md reading Q20) -------------------------------
def sh32_scales(sh: np.ndarray) -> np.ndarray:
    """Per-(basis, channel) scale table [16][3] (Y, Co, Cg): |v| at sorted index floor(0.999 N), the maximum for the DC basis."""
    sh = np.ascontiguousarray(sh, np.float32)
    assert sh.shape[1:] == (16, 3)
    out = np.zeros((16, 3), np.float32)
    lib().orc_sh32_scales(sh.shape[0], _p(sh, C.c_float), _p(out, C.c_float))
    return out


def sh32_encode(sh: np.ndarray, scales: np.ndarray) -> np.ndarray:
    sh = np.ascontiguousarray(sh, np.float32); scales = np.ascontiguousarray(scales, np.float32)
    out = np.zeros((sh.shape[0], 32), np.uint8)
    lib().orc_sh32_encode(sh.shape[0], _p(sh, C.c_float), _p(scales, C.c_float), _p(out, C.c_uint8))
    return out


def sh32_decode(codes: np.ndarray, scales: np.ndarray) -> np.ndarray:
    codes = np.ascontiguousarray(codes, np.uint8); scales = np.ascontiguousarray(scales, np.float32)
    out = np.zeros((codes.shape[0], 16, 3), np.float32)
    lib().orc_sh32_decode(codes.shape[0], _p(codes, C.c_uint8), _p(scales, C.c_float), _p(out, C.c_float))
    return out

"""Seeded synthetic scene + camera generators for the HiGS forward render path.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the
CUDA path (``paper_2606_00352_b200/``).  It holds none of the method's
arithmetic: it only draws random gaussian parameters and builds pinhole
cameras.  Everything is numpy, seeded with ``PCG64(1000 + cfg)``.

The five configurations are the ones BASELINE.json ``configs`` lists; they
stand in for the paper's Mip-NeRF 360 / Inria-model scenes (§5.1:
1.2-6.1 M gaussians, SH degree 3, 1080p and 4K), which are not available here.
The recipe (cluster placement, orbit formulas, ...) is stated in DESIGN.md §4.

Conventions:
  * inputs are *activated*: linear scales (>0), opacities in (0,1);
  * quaternions are (w, x, y, z), not normalised;
  * SH is [N][K][3] with K = (degree+1)^2;
  * camera frame: +x right, +y down, +z forward; ``view`` is the row-major 3x4
    world->camera matrix [R|t]; pixel (i, j) has its centre at (i+0.5, j+0.5).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List

import numpy as np

SH_C0 = 0.28209479177387814  # 1/(2 sqrt(pi)); only used to place the DC colour in U(0,1)


@dataclass
class Camera:
    view: np.ndarray          # (12,) float32 row-major 3x4 [R|t]
    fx: float
    fy: float
    cx: float
    cy: float
    near_z: float
    cam_pos: np.ndarray       # (3,) float32 world-space camera centre
    W: int
    H: int

    def as_floats(self) -> np.ndarray:
        """The 20 floats of the C camera struct: view[12], fx, fy, cx, cy, near_z, cam_pos[3]."""
        out = np.empty(20, dtype=np.float32)
        out[0:12] = self.view
        out[12:16] = (self.fx, self.fy, self.cx, self.cy)
        out[16] = self.near_z
        out[17:20] = self.cam_pos
        return out


@dataclass
class Scene:
    name: str
    means: np.ndarray         # (N,3) float32
    scales: np.ndarray        # (N,3) float32, linear
    quats: np.ndarray         # (N,4) float32, (w,x,y,z), unnormalised
    opacities: np.ndarray     # (N,)  float32 in (0,1)
    sh: np.ndarray            # (N,K,3) float32
    degree: int
    cameras: List[Camera] = field(default_factory=list)

    @property
    def N(self) -> int:
        return int(self.means.shape[0])


def _fov_intrinsics(W: int, H: int, fov_x_deg: float = 60.0):
    fx = (W / 2.0) / np.tan(np.deg2rad(fov_x_deg) / 2.0)
    return float(np.float32(fx)), float(np.float32(fx)), W / 2.0, H / 2.0


def make_camera(W: int, H: int, eye=(0.0, 0.0, 0.0), centre=None, fov_x_deg: float = 60.0,
                near_z: float = 0.2) -> Camera:
    """Pinhole camera; identity pose if ``centre`` is None, else look-at with +y down."""
    fx, fy, cx, cy = _fov_intrinsics(W, H, fov_x_deg)
    eye = np.asarray(eye, dtype=np.float64)
    if centre is None:
        R = np.eye(3)
    else:
        f = np.asarray(centre, dtype=np.float64) - eye
        f /= np.linalg.norm(f)
        down = np.array([0.0, 1.0, 0.0])
        r = np.cross(down, f)
        r /= np.linalg.norm(r)
        d = np.cross(f, r)
        R = np.stack([r, d, f], axis=0)
    t = -R @ eye
    view = np.concatenate([R, t[:, None]], axis=1).astype(np.float32).reshape(12)
    return Camera(view=view, fx=fx, fy=fy, cx=cx, cy=cy, near_z=near_z,
                  cam_pos=eye.astype(np.float32), W=W, H=H)


def _common(rng: np.random.Generator, N: int, log_scale_mu: float, log_scale_sigma: float,
            opacity_sigma: float, degree: int):
    quats = rng.normal(0.0, 1.0, (N, 4)).astype(np.float32)
    scales = np.exp(rng.normal(log_scale_mu, log_scale_sigma, (N, 3))).astype(np.float32)
    logits = rng.normal(0.0, opacity_sigma, N)
    opac = (1.0 / (1.0 + np.exp(-logits))).astype(np.float32)
    K = (degree + 1) ** 2
    sh = np.empty((N, K, 3), dtype=np.float32)
    sh[:, 0, :] = ((rng.random((N, 3)) - 0.5) / SH_C0).astype(np.float32)
    if K > 1:
        # drawn in slabs to keep the float64 temporaries small at 5.8 M gaussians
        step = 1 << 20
        for s in range(0, N, step):
            e = min(N, s + step)
            sh[s:e, 1:, :] = rng.normal(0.0, 0.1, (e - s, K - 1, 3)).astype(np.float32)
    return quats, scales, opac, sh


def scene_cfg0(N: int = 1000, W: int = 128, H: int = 128, seed: int = 1000) -> Scene:
    """Tiny scene: uniform box in front of an identity-pose camera, SH degree 0."""
    rng = np.random.Generator(np.random.PCG64(seed))
    means = np.empty((N, 3), dtype=np.float32)
    means[:, 0] = rng.uniform(-1, 1, N)
    means[:, 1] = rng.uniform(-1, 1, N)
    means[:, 2] = rng.uniform(2, 4, N)
    quats, scales, opac, sh = _common(rng, N, -3.5, 0.5, 1.5, 0)
    return Scene("cfg0_tiny", means, scales, quats, opac, sh, 0, [make_camera(W, H)])


def scene_cfg1(N: int = 100_000, W: int = 640, H: int = 480, seed: int = 1001) -> Scene:
    """Small scene: 16 isotropic clusters (sigma 0.3) in a 4x4x4 box 3 units ahead, SH degree 3."""
    rng = np.random.Generator(np.random.PCG64(seed))
    centres = np.stack([rng.uniform(-2, 2, 16), rng.uniform(-2, 2, 16), rng.uniform(3, 7, 16)], axis=1)
    which = rng.integers(0, 16, N)
    means = (centres[which] + rng.normal(0.0, 0.3, (N, 3))).astype(np.float32)
    quats, scales, opac, sh = _common(rng, N, -4.0, 0.6, 1.5, 3)
    return Scene("cfg1_small", means, scales, quats, opac, sh, 3, [make_camera(W, H)])


def scene_cfg2(N: int = 1_000_000, W: int = 1920, H: int = 1080, seed: int = 1002,
               n_views: int = 8) -> Scene:
    """Medium scene with hotspots: 70 % in 8 tight clusters, 30 % uniform; 8 orbit poses."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n_cl = int(round(0.7 * N))
    centres = rng.uniform(-3, 3, (8, 3))
    sig = rng.uniform(0.05, 0.2, 8)
    which = rng.integers(0, 8, n_cl)
    cl = centres[which] + rng.normal(0.0, 1.0, (n_cl, 3)) * sig[which][:, None]
    un = rng.uniform(-5, 5, (N - n_cl, 3))
    means = np.concatenate([cl, un], axis=0).astype(np.float32)
    quats, scales, opac, sh = _common(rng, N, -4.5, 0.8, 1.5, 3)
    cams = []
    for k in range(n_views):
        th = 2.0 * np.pi * k / n_views
        eye = (6.0 * np.sin(th), 0.0, -6.0 * np.cos(th))
        cams.append(make_camera(W, H, eye=eye, centre=(0.0, 0.0, 0.0)))
    return Scene("cfg2_medium", means, scales, quats, opac, sh, 3, cams)


def _random_rotations(rng: np.random.Generator, n: int) -> np.ndarray:
    q = rng.normal(0.0, 1.0, (n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((n, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - w * z); R[:, 0, 2] = 2 * (x * z + w * y)
    R[:, 1, 0] = 2 * (x * y + w * z); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - w * x)
    R[:, 2, 0] = 2 * (x * z - w * y); R[:, 2, 1] = 2 * (y * z + w * x); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def orbit_cameras(W: int, H: int, n_views: int = 32) -> List[Camera]:
    """cfg3/cfg4 orbit: radius 6.5 + 1.5 sin 2θ in [5, 8], elevation 20° sin 3θ, look at origin."""
    cams = []
    for k in range(n_views):
        th = 2.0 * np.pi * k / n_views
        r = 6.5 + 1.5 * np.sin(2 * th)
        el = np.deg2rad(20.0) * np.sin(3 * th)
        eye = (r * np.cos(el) * np.sin(th), -r * np.sin(el), -r * np.cos(el) * np.cos(th))
        cams.append(make_camera(W, H, eye=eye, centre=(0.0, 0.0, 0.0)))
    return cams


def scene_large(N: int = 5_800_000, W: int = 1920, H: int = 1080, seed: int = 1003,
                n_views: int = 32) -> Scene:
    """Large, paper-scale scene: heavy-tailed density on 200 planes / ellipsoid shells,
    20 % uniform background, 10 % in one hot region.  cfg3 = this at 1080p (view 0),
    cfg4 = the same arrays at 3840x2160 over the 32-view orbit."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n_surf = int(round(0.7 * N))
    n_bg = int(round(0.2 * N))
    n_hot = N - n_surf - n_bg
    S = 200
    wts = rng.pareto(1.5, S) + 0.05
    wts /= wts.sum()
    which = rng.choice(S, size=n_surf, p=wts)
    centres = rng.uniform(-4, 4, (S, 3))
    rots = _random_rotations(rng, S)
    ext = rng.uniform(0.3, 2.0, (S, 3))
    is_plane = np.arange(S) < (S // 2)
    local = np.empty((n_surf, 3))
    uv = rng.uniform(-1, 1, (n_surf, 2))
    dirs = rng.normal(0.0, 1.0, (n_surf, 3))
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    pl = is_plane[which]
    local[pl, 0] = uv[pl, 0]; local[pl, 1] = uv[pl, 1]; local[pl, 2] = 0.0
    local[~pl] = dirs[~pl]
    local *= ext[which]
    surf = np.einsum("nij,nj->ni", rots[which], local) + centres[which] + rng.normal(0.0, 0.01, (n_surf, 3))
    bg = rng.uniform(-6, 6, (n_bg, 3))
    hot = np.array([0.5, 0.2, 0.0]) + rng.normal(0.0, 0.15, (n_hot, 3))
    means = np.concatenate([surf, bg, hot], axis=0)
    # trained 3DGS models are not stored in generation order; shuffle so ids carry no structure
    perm = rng.permutation(N)
    means = means[perm].astype(np.float32)
    quats, scales, opac, sh = _common(rng, N, -5.0, 1.0, 2.0, 3)
    return Scene(f"large_{N}", means, scales, quats, opac, sh, 3, orbit_cameras(W, H, n_views))


def scene_cfg3(N: int = 5_800_000) -> Scene:
    s = scene_large(N, 1920, 1080)
    s.name = "cfg3_large_1080p"
    return s


def scene_cfg4(N: int = 5_800_000) -> Scene:
    s = scene_large(N, 3840, 2160)
    s.name = "cfg4_large_4k"
    return s


def retarget(scene: Scene, W: int, H: int) -> Scene:
    """Same gaussians and poses, cameras rebuilt for another resolution (fov_x stays 60 deg)."""
    cams = []
    for c in scene.cameras:
        fx, fy, cx, cy = _fov_intrinsics(W, H)
        cams.append(Camera(view=c.view.copy(), fx=fx, fy=fy, cx=cx, cy=cy, near_z=c.near_z,
                           cam_pos=c.cam_pos.copy(), W=W, H=H))
    return Scene(scene.name, scene.means, scene.scales, scene.quats, scene.opacities, scene.sh,
                 scene.degree, cams)


def single_gaussian(mean, scale, quat=(1, 0, 0, 0), opacity=0.8, rgb=(0.9, 0.5, 0.1), W=129, H=129) -> Scene:
    """One gaussian with a degree-0 colour; used by the closed-form pins."""
    return stack_gaussians([mean], [scale], [quat], [opacity], [rgb], W, H)


def stack_gaussians(means, scales, quats, opacities, rgbs, W=129, H=129) -> Scene:
    """A hand-specified list of degree-0 gaussians seen by an identity-pose camera."""
    means = np.asarray(means, dtype=np.float32).reshape(-1, 3)
    N = means.shape[0]
    scales = np.asarray(scales, dtype=np.float32)
    if scales.ndim == 1:                      # one isotropic scale per gaussian
        scales = np.repeat(scales[:, None], 3, axis=1)
    scales = scales.reshape(N, 3).copy()
    quats = np.asarray(quats, dtype=np.float32).reshape(N, 4)
    opac = np.asarray(opacities, dtype=np.float32).reshape(N)
    rgb = np.asarray(rgbs, dtype=np.float64).reshape(N, 3)
    sh = ((rgb - 0.5) / SH_C0).astype(np.float32).reshape(N, 1, 3)
    return Scene("handmade", means, scales, quats, opac, sh, 0, [make_camera(W, H)])


def needle_scene(n: int = 300, W: int = 1920, H: int = 1080, seed: int = 6, sigma_lo_px: float = 60.0,
                 sigma_hi_px: float = 350.0) -> Scene:
    """Near-camera needles: one long axis (log-uniform screen-space sigma in [lo, hi] px), two axes of 1e-5,
    rotated about the view axis by a random angle, centres spread over the image; degree-0 colours.  The conic
    of such a gaussian is ill-conditioned (a c / det up to 1e5-1e7): the stress case for the conservative
    bounding box / row scan (reading Q8)."""
    rng = np.random.default_rng(seed)
    fx = (W / 2.0) / np.tan(np.pi / 6.0)
    z = rng.uniform(0.5, 1.5, n)
    means = np.stack([rng.uniform(-0.4, 0.4, n) * z, rng.uniform(-0.25, 0.25, n) * z, z], axis=1)
    sig_px = np.exp(rng.uniform(np.log(sigma_lo_px), np.log(sigma_hi_px), n))
    scales = np.stack([sig_px * z / fx, np.full(n, 1e-5), np.full(n, 1e-5)], axis=1)
    th = rng.uniform(0.0, np.pi, n)
    quats = np.stack([np.cos(th / 2), np.zeros(n), np.zeros(n), np.sin(th / 2)], axis=1)
    return stack_gaussians(means, scales, quats, rng.uniform(0.3, 0.99, n), rng.uniform(0, 1, (n, 3)), W, H)


CONFIGS = {0: scene_cfg0, 1: scene_cfg1, 2: scene_cfg2, 3: scene_cfg3, 4: scene_cfg4}


def make_scene(cfg: int, **kw) -> Scene:
    return CONFIGS[cfg](**kw)

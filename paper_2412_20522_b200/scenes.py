"""Seeded synthetic scene generators (inputs only -- none of the method's arithmetic).

These stand in for the paper's datasets (Mip-NeRF360, Tanks & Temples, Deep Blending;
PAPER.md:130, section 4.1), which are not available.  Gaussian counts and image sizes are
BASELINE.json's `configs` (3 M ~ the unpruned Mip-NeRF360 average, Tab. 1;
6 M ~ the largest scenes, Tab. 12).  The recipe is in DESIGN.md "Input recipe".

The SAME fp32 arrays produced here are given to the CPU oracle (`oracle/`) and to the CUDA
library (`paper_2412_20522_b200.binding`).  This module imports neither of them.

Draw order per scene (numpy `default_rng(seed)`): means, log-scales, quaternions, opacity
logits, SH, mask keep-probabilities, mask uniforms, upstream image gradient.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np


@dataclass
class Camera:
    """Pinhole camera.  x_cam = R @ x_world + t; looks down +z, x right, y down."""

    width: int
    height: int
    fx: float
    fy: float
    cx: float
    cy: float
    R: np.ndarray  # 3x3 row-major, float64
    t: np.ndarray  # 3, float64
    bg: tuple = (0.0, 0.0, 0.0)
    sh_degree: int = 0


@dataclass
class Scene:
    name: str
    means: np.ndarray  # N x 3 fp32 (world space)
    log_scales: np.ndarray  # N x 3 fp32
    quats: np.ndarray  # N x 4 fp32 (w, x, y, z), not necessarily unit
    opacity_logits: np.ndarray  # N fp32
    sh: np.ndarray  # N x K x 3 fp32
    masks: np.ndarray  # N fp32 in {0, 1}
    cameras: list = field(default_factory=list)
    seed: int = 0

    @property
    def N(self) -> int:
        return int(self.means.shape[0])

    @property
    def camera(self) -> Camera:
        return self.cameras[0]

    def dL_dimage(self, cam_index: int = 0) -> np.ndarray:
        """Upstream gradient ~ N(0,1), planar [3][H][W] fp32, seeded per (scene, camera)."""
        cam = self.cameras[cam_index]
        rng = np.random.default_rng([self.seed, 7919, cam_index])
        return rng.standard_normal((3, cam.height, cam.width), dtype=np.float32)


def look_at(position, target, down=(0.0, 1.0, 0.0)):
    """World->camera (R, t) for a camera at `position` looking at `target`; world 'down' = +y."""
    position = np.asarray(position, np.float64)
    z = np.asarray(target, np.float64) - position
    z /= np.linalg.norm(z)
    x = np.cross(np.asarray(down, np.float64), z)
    x /= np.linalg.norm(x)
    y = np.cross(z, x)
    R = np.stack([x, y, z])
    return R, -R @ position


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _quats(rng, n):
    q = rng.standard_normal((n, 4))
    return q / np.linalg.norm(q, axis=1, keepdims=True)


def _sh(rng, n, degree, dc_sigma=0.5, rest_sigma=0.05):
    K = (degree + 1) ** 2
    sh = np.empty((n, K, 3), np.float32)
    sh[:, 0, :] = rng.standard_normal((n, 3)) * dc_sigma
    if K > 1:
        sh[:, 1:, :] = rng.standard_normal((n, K - 1, 3), dtype=np.float32) * rest_sigma
    return sh


def _masks(rng, n, keep):
    """keep: float (constant probability) or 'uniform' (p_i ~ U(0,1))."""
    p = rng.random(n) if keep == "uniform" else np.full(n, float(keep))
    u = rng.random(n)
    return (u < p).astype(np.float32)


def _fov_focal(width, fov_deg):
    return 0.5 * width / math.tan(math.radians(fov_deg) / 2)


def config1(n=1000, width=128, height=128, seed=0) -> Scene:
    """Tiny scene (BASELINE.json configs[0]): camera-space means, SH degree 0."""
    rng = np.random.default_rng(seed)
    means = np.column_stack([rng.uniform(-1, 1, n), rng.uniform(-1, 1, n), rng.uniform(2, 6, n)])
    log_scales = rng.normal(-3.5, 0.5, (n, 3))
    quats = _quats(rng, n)
    logits = rng.normal(0, 1, n)
    sh = _sh(rng, n, 0)
    masks = _masks(rng, n, 0.5)
    cam = Camera(width, height, 120.0 * width / 128, 120.0 * width / 128, width / 2, height / 2,
                 np.eye(3), np.zeros(3), sh_degree=0)
    return Scene("cfg1_tiny", _f32(means), _f32(log_scales), _f32(quats), _f32(logits), sh, masks, [cam], seed)


def config2(n=100_000, width=512, height=512, seed=1) -> Scene:
    """Small scene (configs[1]): 64 isotropic clusters, camera at distance 6, FOV 60, SH degree 3."""
    rng = np.random.default_rng(seed)
    centres = rng.uniform(-3, 3, (64, 3))
    pick = rng.integers(0, 64, n)
    means = centres[pick] + rng.normal(0, 0.3, (n, 3))
    log_scales = rng.normal(-4.0, 0.7, (n, 3))
    quats = _quats(rng, n)
    logits = rng.normal(0, 1.5, n)
    sh = _sh(rng, n, 3)
    masks = _masks(rng, n, 0.4)
    R, t = look_at((0, 0, -6), (0, 0, 0))
    f = _fov_focal(width, 60)
    cam = Camera(width, height, f, f, width / 2, height / 2, R, t, sh_degree=3)
    return Scene("cfg2_small", _f32(means), _f32(log_scales), _f32(quats), _f32(logits), sh, masks, [cam], seed)


def _outdoor_geometry(rng, n):
    n_fg = int(round(0.8 * n))
    n_bg = n - n_fg
    # 256 cluster centres uniform in the ball of radius 4
    v = rng.standard_normal((256, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    centres = v * (4.0 * rng.random(256) ** (1 / 3))[:, None]
    fg = centres[rng.integers(0, 256, n_fg)] + rng.normal(0, 0.25, (n_fg, 3))
    d = rng.standard_normal((n_bg, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    bg = d * rng.uniform(20, 100, n_bg)[:, None]
    means = np.concatenate([fg, bg])
    log_scales = np.concatenate([rng.normal(-4.5, 0.8, (n_fg, 3)), rng.normal(-1.0, 0.8, (n_bg, 3))])
    return means, log_scales


def config3(n=3_000_000, width=1297, height=840, seed=2, keep="uniform", n_cameras=1, radius=8.0) -> Scene:
    """Unbounded outdoor-shaped scene (configs[2]): 80% foreground clusters, 20% background shell."""
    rng = np.random.default_rng(seed)
    means, log_scales = _outdoor_geometry(rng, n)
    quats = _quats(rng, n)
    logits = rng.normal(0, 2.0, n)
    sh = _sh(rng, n, 3)
    masks = _masks(rng, n, keep)
    f = _fov_focal(width, 60)
    cams = []
    for k in range(n_cameras):
        th = 2 * math.pi * k / max(n_cameras, 1)
        R, t = look_at((radius * math.sin(th), 0.0, -radius * math.cos(th)), (0, 0, 0))
        cams.append(Camera(width, height, f, f, width / 2, height / 2, R, t, sh_degree=3))
    return Scene("cfg3_outdoor", _f32(means), _f32(log_scales), _f32(quats), _f32(logits), sh, masks, cams, seed)


def config4(n=2_800_000, width=1264, height=832, seed=3) -> Scene:
    """Indoor-shaped scene (configs[3]): box walls + 30 furniture clusters, camera inside, FOV 70."""
    rng = np.random.default_rng(seed)
    n_wall = int(round(0.7 * n))
    n_cl = n - n_wall
    half = np.array([5.0, 2.0, 3.0])
    # area-weighted face choice: faces normal to x (area 4x6), y (10x6), z (10x4)
    areas = np.array([4 * 6, 4 * 6, 10 * 6, 10 * 6, 10 * 4, 10 * 4], np.float64)
    face = rng.choice(6, n_wall, p=areas / areas.sum())
    pts = rng.uniform(-1, 1, (n_wall, 3)) * half
    axis = face // 2
    sign = np.where(face % 2 == 0, -1.0, 1.0)
    pts[np.arange(n_wall), axis] = sign * half[axis]
    centres = rng.uniform(-0.9, 0.9, (30, 3)) * half
    cl = centres[rng.integers(0, 30, n_cl)] + rng.normal(0, 0.2, (n_cl, 3))
    means = np.concatenate([pts, cl])
    log_scales = rng.normal(-4.0, 0.6, (n, 3))
    quats = _quats(rng, n)
    logits = rng.normal(0.5, 1.5, n)
    sh = _sh(rng, n, 3)
    masks = _masks(rng, n, 0.35)
    R, t = look_at((-3, 0, 0), (5, 0, 0))
    f = _fov_focal(width, 70)
    cam = Camera(width, height, f, f, width / 2, height / 2, R, t, sh_degree=3)
    return Scene("cfg4_indoor", _f32(means), _f32(log_scales), _f32(quats), _f32(logits), sh, masks, [cam], seed)


def config5(n=6_000_000, width=1920, height=1080, seed=4, n_cameras=20) -> Scene:
    """Stress scene (configs[4]): generator of config 3, keep-probability 0.9, 20 cameras on a circle."""
    s = config3(n, width, height, seed, keep=0.9, n_cameras=n_cameras)
    s.name = "cfg5_stress"
    return s


def tiny_fd_scene(n=8, width=32, height=32, seed=100, sh_degree=3, bg=(0.2, 0.5, 0.7)) -> Scene:
    """A few large-ish overlapping Gaussians for finite-difference pins."""
    rng = np.random.default_rng(seed)
    means = np.column_stack([rng.uniform(-0.8, 0.8, n), rng.uniform(-0.8, 0.8, n), rng.uniform(-1.0, 1.0, n)])
    log_scales = rng.normal(-1.6, 0.4, (n, 3))
    quats = rng.standard_normal((n, 4)) * 1.3  # deliberately not unit
    logits = rng.normal(0.5, 1.5, n)
    logits[0] = 7.0  # opacity ~ 0.999: exercises the 0.99 clamp
    sh = _sh(rng, n, sh_degree, 0.5, 0.2)
    masks = _masks(rng, n, 0.5)
    masks[0] = 1.0
    R, t = look_at((0.3, -0.2, -4.0), (0, 0, 0))
    f = _fov_focal(width, 50)
    cam = Camera(width, height, f, 1.1 * f, width / 2 + 0.7, height / 2 - 0.4, R, t, bg=bg, sh_degree=sh_degree)
    return Scene("tiny_fd", _f32(means), _f32(log_scales), _f32(quats), _f32(logits), sh, masks, [cam], seed)


def needles(n=4000, width=640, height=400, seed=11) -> Scene:
    """Long thin splats seen far from their centres (real captures are full of them; configs 1-5 have few): one axis
    30-300x the other two, random orientation, so that the three terms of the exponent reach 1e4..1e6 at pixels that
    still pass the alpha filter and cancel there."""
    rng = np.random.default_rng(seed)
    means = np.column_stack([rng.uniform(-2.5, 2.5, n), rng.uniform(-1.5, 1.5, n), rng.uniform(-1.0, 1.0, n)])
    log_scales = rng.normal(-6.0, 0.5, (n, 3))
    log_scales[np.arange(n), rng.integers(0, 3, n)] = rng.normal(-1.0, 0.6, n)
    quats = _quats(rng, n)
    logits = rng.normal(1.0, 1.5, n)
    sh = _sh(rng, n, 1)
    masks = _masks(rng, n, 0.6)
    R, t = look_at((0.0, 0.0, -5.0), (0, 0, 0))
    f = _fov_focal(width, 55)
    cam = Camera(width, height, f, f, width / 2, height / 2, R, t, sh_degree=1)
    return Scene("needles", _f32(means), _f32(log_scales), _f32(quats), _f32(logits), sh, masks, [cam], seed)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def make(config: int, **kw) -> Scene:
    return CONFIGS[config](**kw)


def mask_head_inputs(n, seed=7, n_draws=10, score_sigma=2.0):
    """Seeded inputs of the mask head: 2 scores per Gaussian and the uniforms its samplers
    consume (one draw for the training sample, n_draws for the prune rule).  No arithmetic of the method here, and
    no narrowing of the inputs either: the fp32 cast of a uniform on [0,1) can be exactly 0 or exactly 1, and what
    the samplers do with such a value is defined by the method's side (include/mg.h, reading 29)."""
    rng = np.random.default_rng(seed)
    scores = _f32(rng.normal(0.0, score_sigma, (n, 2)))
    u = _f32(rng.uniform(0.0, 1.0, (n, 2)))
    u_prune = _f32(rng.uniform(0.0, 1.0, (n_draws, n, 2)))
    dL_dmask = _f32(rng.normal(0.0, 1.0, n))
    return scores, u, u_prune, dL_dmask

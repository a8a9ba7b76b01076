"""Seeded synthetic inputs for the TurboGS sparse-raster hot path.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2606_15924_b200/``).  It holds no arithmetic of the method: it only
draws random Gaussians, cameras, error maps and targets with the shapes, sizes
and value distributions of BASELINE.json's five configs (the recipe is restated
in DESIGN.md §"Input recipe"; the paper's own datasets -- PAPER.md:263 -- are not
available, these inputs stand in for them).

Everything is NumPy, float32 on output, ``np.random.default_rng(seed)``.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Tuple

import numpy as np

# 1/(2*sqrt(pi)): only used to turn the "RGB ~ U[0,1]" wording of config 1 into a
# degree-0 coefficient (an input convention, not part of the rasteriser).
_DC_SCALE = 0.28209479177387814

TILE = 16
PIXEL_MODE_ALL = 0
PIXEL_MODE_BERNOULLI_ERR = 1


@dataclass
class Camera:
    width: int
    height: int
    fx: float
    fy: float
    cx: float
    cy: float
    R: np.ndarray  # [3,3] world->camera rotation, row-major, float32
    t: np.ndarray  # [3] world->camera translation, float32
    znear: float = 0.2
    bg: Tuple[float, float, float] = (0.0, 0.0, 0.0)

    @property
    def grid(self) -> Tuple[int, int]:
        return ((self.width + TILE - 1) // TILE, (self.height + TILE - 1) // TILE)

    @property
    def num_tiles(self) -> int:
        gx, gy = self.grid
        return gx * gy


@dataclass
class Scene:
    """One workload: Gaussians (activated parameters), a camera and a sampling request."""
    name: str
    cam: Camera
    sh_degree: int
    means3D: np.ndarray    # [N,3]
    scales: np.ndarray     # [N,3]  > 0   (already exp'ed)
    quats: np.ndarray      # [N,4]  wxyz, unit norm
    opacities: np.ndarray  # [N]    in (0,1) (already sigmoid'ed)
    sh: np.ndarray         # [N,K,3]
    # sampling request
    tile_pct: Tuple[int, int]           # (num, den): fraction of tiles to sample
    pixel_mode: int                      # PIXEL_MODE_*
    pix_rate: Tuple[int, int] = (1, 1)  # (num, den) for BERNOULLI_ERR
    sample_seed: int = 0
    err: np.ndarray | None = None        # [H,W] error map, or None => residual of render vs target
    target: np.ndarray | None = None     # [H,W,3] (config 1)
    extra: Dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.means3D.shape[0])


def _unit_quats(rng: np.random.Generator, n: int) -> np.ndarray:
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    return q.astype(np.float32)


def _sigmoid(x):
    return 1.0 / (1.0 + np.exp(-x))


def _sh_deg3(rng: np.random.Generator, n: int) -> np.ndarray:
    sh = rng.normal(0.0, 0.2, size=(n, 16, 3))
    sh[:, 0, :] = rng.normal(0.5, 0.2, size=(n, 3))
    return sh.astype(np.float32)


def blob_error_map(rng: np.random.Generator, width: int, height: int, n_blobs: int) -> np.ndarray:
    """Smooth non-negative error map: a sum of ``n_blobs`` isotropic 2D bumps.

    centres ~ U(image), sigma ~ U[2%,15%] of the image diagonal, amplitude ~ U[0.1,1].
    """
    diag = float(np.hypot(width, height))
    cx = rng.uniform(0, width, n_blobs)
    cy = rng.uniform(0, height, n_blobs)
    sg = rng.uniform(0.02, 0.15, n_blobs) * diag
    am = rng.uniform(0.1, 1.0, n_blobs)
    xs = np.arange(width, dtype=np.float64)[None, :]
    ys = np.arange(height, dtype=np.float64)[:, None]
    e = np.zeros((height, width), dtype=np.float64)
    for b in range(n_blobs):
        e += am[b] * np.exp(-((xs - cx[b]) ** 2 + (ys - cy[b]) ** 2) / (2.0 * sg[b] ** 2))
    return e.astype(np.float32)


def _front_camera(width, height, f, dist) -> Camera:
    """Camera at (0,0,-dist) looking down +z: R = I, t = (0,0,dist)."""
    return Camera(width, height, float(f), float(f), width / 2.0, height / 2.0,
                  np.eye(3, dtype=np.float32), np.array([0, 0, dist], dtype=np.float32))


def orbit_view(scene: "Scene", view: int) -> "Scene":
    """View `view` of a scene whose camera orbits the origin at the scene's distance: view 0 is the scene's own camera,
    view r > 0 is turned by a seeded yaw in [-pi, pi) and pitch in [-0.3, 0.3] about the scene's centre (the Gaussian
    clouds of configs 2-5 are centred there), keeping the distance.  Used by the N > 1 replicas: one view per rank
    (PAPER.md:113).  Input generation only: no arithmetic of the method."""
    if view == 0:
        return scene
    rng = np.random.default_rng(30_000 + int(view))
    yaw, pitch = rng.uniform(-np.pi, np.pi), rng.uniform(-0.3, 0.3)
    cy, sy, cp, sp = np.cos(yaw), np.sin(yaw), np.cos(pitch), np.sin(pitch)
    Ry = np.array([[cy, 0, sy], [0, 1, 0], [-sy, 0, cy]])
    Rx = np.array([[1, 0, 0], [0, cp, -sp], [0, sp, cp]])
    c = scene.cam
    R = (np.asarray(c.R, np.float64) @ Rx @ Ry).astype(np.float32)  # x_cam = R x_world + t with the same t: same distance
    cam = Camera(c.width, c.height, c.fx, c.fy, c.cx, c.cy, R, c.t.copy(), c.znear, c.bg)
    return Scene(f"{scene.name}_view{view}", cam, scene.sh_degree, scene.means3D, scene.scales, scene.quats, scene.opacities,
                 scene.sh, scene.tile_pct, scene.pixel_mode, scene.pix_rate, scene.sample_seed + int(view), scene.err,
                 scene.target, dict(scene.extra))


def config1(seed: int = 0, n: int = 1024) -> Scene:
    """Tiny scene (BASELINE.json configs[0])."""
    rng = np.random.default_rng(seed)
    mu = rng.uniform(-1, 1, size=(n, 3))
    mu[:, 2] += 4.0
    s = np.exp(rng.normal(-3.0, 0.5, size=(n, 3)))
    q = _unit_quats(rng, n)
    o = _sigmoid(rng.normal(0.0, 1.0, size=n))
    rgb = rng.uniform(0, 1, size=(n, 3))
    sh = ((rgb - 0.5) / _DC_SCALE)[:, None, :]
    cam = Camera(128, 128, 128.0, 128.0, 64.0, 64.0, np.eye(3, dtype=np.float32),
                 np.zeros(3, dtype=np.float32))
    target = np.random.default_rng(0).uniform(0, 1, size=(128, 128, 3)).astype(np.float32)
    return Scene("cfg1_tiny", cam, 0, mu.astype(np.float32), s.astype(np.float32), q,
                 o.astype(np.float32), sh.astype(np.float32), (25, 100), PIXEL_MODE_ALL,
                 target=target, sample_seed=seed)


def _gauss_scene(name, seed, n, mean_sigma, log_scale, opac_sigma, width, height, f, dist,
                 n_blobs, tile_pct, pixel_mode, pix_rate=(1, 1), clusters=False) -> Scene:
    rng = np.random.default_rng(seed)
    mu = rng.normal(0.0, mean_sigma, size=(n, 3))
    if clusters:
        # 20% of the Gaussians re-drawn around 8 tight clusters (sigma 0.1) -> tile-load imbalance
        n_c = n // 5
        centres = rng.normal(0.0, mean_sigma, size=(8, 3))
        which = rng.integers(0, 8, size=n_c)
        idx = rng.permutation(n)[:n_c]
        mu[idx] = centres[which] + rng.normal(0.0, 0.1, size=(n_c, 3))
    s = np.exp(rng.normal(log_scale[0], log_scale[1], size=(n, 3)))
    q = _unit_quats(rng, n)
    o = _sigmoid(rng.normal(0.0, opac_sigma, size=n))
    sh = _sh_deg3(rng, n)
    cam = _front_camera(width, height, f, dist)
    err = blob_error_map(rng, width, height, n_blobs)
    return Scene(name, cam, 3, mu.astype(np.float32), s.astype(np.float32), q,
                 o.astype(np.float32), sh, tile_pct, pixel_mode, pix_rate, sample_seed=seed,
                 err=err)


def config2(seed: int = 1, n: int = 100_000) -> Scene:
    """100k Gaussians, 980x545, top 30% tiles, all pixels (configs[1], the bench workload)."""
    return _gauss_scene("cfg2_100k", seed, n, np.sqrt(2.0), (-4.0, 0.7), 1.5, 980, 545, 900.0, 6.0,
                        32, (30, 100), PIXEL_MODE_ALL)


def config3(seed: int = 2, n: int = 1_000_000) -> Scene:
    """1M Gaussians with 8 tight clusters, 1600x1063, 20% tiles, Bernoulli(1/2) pixels."""
    return _gauss_scene("cfg3_1M_clustered", seed, n, 2.0, (-4.0, 0.7), 1.5, 1600, 1063, 1400.0, 8.0,
                        32, (20, 100), PIXEL_MODE_BERNOULLI_ERR, (1, 2), clusters=True)


def config4(seed: int = 3, n: int = 3_000_000) -> Scene:
    """3M Gaussians, 1957x1091, dense mask (100% tiles, all pixels)."""
    return _gauss_scene("cfg4_3M_dense", seed, n, np.sqrt(6.0), (-4.5, 0.8), 2.0, 1957, 1091, 1700.0,
                        12.0, 32, (100, 100), PIXEL_MODE_ALL)


def config5(pct: int = 20, seed: int = 4, n: int = 1_000_000) -> Scene:
    """Sampling-rate sweep: 1M Gaussians, 1297x840, pct in {5,10,20,40,70,100}."""
    sc = _gauss_scene(f"cfg5_1M_pct{pct}", seed, n, 2.0, (-4.0, 0.7), 1.5, 1297, 840, 1100.0, 8.0,
                      64, (pct, 100), PIXEL_MODE_ALL)
    return sc


SWEEP_PCTS = (5, 10, 20, 40, 70, 100)


def make(config: int, **kw) -> Scene:
    """``config`` is 1-based, as in BASELINE.json's prose ("config 1" == configs[0])."""
    return {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}[config](**kw)


def dl_dcolor(seed: int, n: int) -> np.ndarray:
    """Seeded upstream gradient dL/dcolor [n,3] ~ N(0,1) for parity runs (an input of the
    backward pass; the loss itself is outside the hot path)."""
    return np.random.default_rng(10_000 + seed).standard_normal((n, 3)).astype(np.float32)


def small_random_scene(seed: int, n: int, width: int, height: int, sh_degree: int = 3,
                       f: float | None = None, dist: float = 4.0, rotate: bool = True,
                       bg=(0.0, 0.0, 0.0), spread: float = 1.0, log_scale=(-2.5, 0.5)) -> Scene:
    """Small general-position scene (rotated camera, non-zero background) for tests."""
    rng = np.random.default_rng(seed)
    K = (sh_degree + 1) ** 2
    mu = rng.uniform(-spread, spread, size=(n, 3))
    s = np.exp(rng.normal(log_scale[0], log_scale[1], size=(n, 3)))
    q = _unit_quats(rng, n)
    o = _sigmoid(rng.normal(0.0, 1.0, size=n))
    sh = rng.normal(0.0, 0.3, size=(n, K, 3))
    sh[:, 0, :] = rng.normal(0.3, 0.5, size=(n, 3))
    if f is None:
        f = float(max(width, height))
    if rotate:
        # small random rotation about a random axis (Rodrigues), camera still sees the origin
        ax = rng.standard_normal(3)
        ax /= np.linalg.norm(ax)
        ang = rng.uniform(-0.3, 0.3)
        Kx = np.array([[0, -ax[2], ax[1]], [ax[2], 0, -ax[0]], [-ax[1], ax[0], 0]])
        R = np.eye(3) + np.sin(ang) * Kx + (1 - np.cos(ang)) * (Kx @ Kx)
    else:
        R = np.eye(3)
    t = np.array([0.0, 0.0, dist]) + (rng.uniform(-0.1, 0.1, 3) if rotate else 0.0)
    cam = Camera(width, height, float(f), float(f), width / 2.0, height / 2.0,
                 R.astype(np.float32), t.astype(np.float32), 0.2, tuple(float(b) for b in bg))
    err = blob_error_map(rng, width, height, 6)
    return Scene(f"small_{seed}", cam, sh_degree, mu.astype(np.float32), s.astype(np.float32), q,
                 o.astype(np.float32), sh.astype(np.float32), (50, 100), PIXEL_MODE_ALL,
                 sample_seed=seed, err=err)


# ---- inputs of the moment-damped LM solve (no method arithmetic here) --------
LM_KEYS = ("means3D", "scales", "quats", "opacities", "sh")
_LM_SHAPES = {"means3D": (3,), "scales": (3,), "quats": (4,), "opacities": ()}
# typical magnitudes of one view's per-Gaussian gradients in a 3DGS run (activated parameters)
_LM_SIGMA = {"means3D": 2e-3, "scales": 5e-3, "quats": 1e-3, "opacities": 1e-2, "sh": 3e-3}


def lm_state(seed: int, n: int, sh_degree: int = 3, views: int = 1, p_update: float = 0.7, warm: bool = True):
    """Seeded optimiser state for `tgs_lm_solve`: per-view gradients [V, N, ...] (heavy tailed: N(0, sigma) times a
    per-Gaussian log-normal factor; Gaussians outside `update` have zero gradients, as the sparse raster backward
    leaves them), Adam moments m, v in the parameter layouts (warm: as after some iterations; cold: zeros) and
    the update mask (int32, 1 = received a gradient).  Returns (grads, m, v, update), dicts keyed by LM_KEYS."""
    rng = np.random.default_rng(20_000 + seed)
    K = (sh_degree + 1) ** 2
    shapes = dict(_LM_SHAPES, sh=(K, 3))
    update = (rng.random(n) < p_update).astype(np.int32)
    if n > 0:
        update[0] = 1
    boost = np.exp(rng.normal(0.0, 1.0, size=n))
    grads, m, v = {}, {}, {}
    for key in LM_KEYS:
        shp = shapes[key]
        ex = (slice(None),) + (None,) * len(shp)
        sig = _LM_SIGMA[key]
        g = rng.standard_normal((views, n) + shp) * sig
        g *= (boost * update)[(None,) + ex]
        if key == "sh":
            g[:, :, 0, :] *= 3.0  # the DC band carries the larger gradient
        grads[key] = g.astype(np.float32)
        if warm:
            m[key] = (rng.standard_normal((n,) + shp) * 0.5 * sig * boost[ex]).astype(np.float32)
            v[key] = ((0.05 + rng.random((n,) + shp)) * (sig * boost[ex]) ** 2).astype(np.float32)
        else:
            m[key] = np.zeros((n,) + shp, np.float32)
            v[key] = np.zeros((n,) + shp, np.float32)
    return grads, m, v, update

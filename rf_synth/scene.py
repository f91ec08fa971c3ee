"""Analytic scenes: an axis-aligned box room seen from inside plus spheres and axis-aligned boxes.

Stand-in for the paper's room-scale sequences (FastCaMo-Synth / ICL-NUIM), which
are not available; only shapes (room scale, object sizes) are taken.  SURVEY.md 8(d), A24.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class Scene:
    room_lo: np.ndarray                      # (3,) inner room faces, metres
    room_hi: np.ndarray                      # (3,)
    spheres: np.ndarray = field(default_factory=lambda: np.zeros((0, 4)))   # (n,4) cx,cy,cz,r
    boxes: np.ndarray = field(default_factory=lambda: np.zeros((0, 6)))     # (n,6) cx,cy,cz,hx,hy,hz


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(int(seed)))


def make_scene(seed: int, extent: float, inset: float, n_spheres: int, n_boxes: int,
               clearance: float = 0.3) -> Scene:
    """Room of volume extent `extent` whose inner faces are inset by `inset`, with
    seeded spheres (r in [0.1,0.3] m) and axis-aligned boxes (side in [0.2,0.6] m) whose centres
    keep `clearance` from the walls."""
    rng = _rng(seed)
    lo = np.full(3, inset, dtype=np.float64)
    hi = np.full(3, extent - inset, dtype=np.float64)
    sph = np.zeros((n_spheres, 4))
    for i in range(n_spheres):
        r = rng.uniform(0.1, 0.3)
        c = rng.uniform(lo + clearance, hi - clearance)
        sph[i] = (*c, r)
    box = np.zeros((n_boxes, 6))
    for i in range(n_boxes):
        h = rng.uniform(0.1, 0.3, size=3)
        c = rng.uniform(lo + clearance, hi - clearance)
        box[i] = (*c, *h)
    return Scene(lo, hi, sph, box)


def _sd_box(p: np.ndarray, c: np.ndarray, h: np.ndarray) -> np.ndarray:
    """Exact signed distance to an axis-aligned box (negative inside)."""
    q = np.abs(p - c) - h
    outside = np.linalg.norm(np.maximum(q, 0.0), axis=-1)
    inside = np.minimum(np.max(q, axis=-1), 0.0)
    return outside + inside


def scene_sdf(scene: Scene, p: np.ndarray) -> np.ndarray:
    """Signed distance of the free space boundary: positive in free space, negative inside walls
    and objects.  p: (...,3)."""
    p = np.asarray(p, dtype=np.float64)
    rc = 0.5 * (scene.room_lo + scene.room_hi)
    rh = 0.5 * (scene.room_hi - scene.room_lo)
    d = -_sd_box(p, rc, rh)
    for s in scene.spheres:
        d = np.minimum(d, np.linalg.norm(p - s[:3], axis=-1) - s[3])
    for b in scene.boxes:
        d = np.minimum(d, _sd_box(p, b[:3], b[3:]))
    return d


def analytic_volume(scene: Scene, dims, voxel_size: float, trunc: float, origin=(0.0, 0.0, 0.0),
                    half: bool = False):
    """clamp(sdf_scene(voxel centre)/trunc, -1, 1) on a dense grid, index x + X*(y + Y*z); W = 1
    everywhere.  With half=True the values are rounded to binary16 (and returned as float32)."""
    X, Y, Z = (int(v) for v in dims)
    out = np.empty((Z, Y, X), dtype=np.float32)
    xs = origin[0] + (np.arange(X) + 0.5) * voxel_size
    ys = origin[1] + (np.arange(Y) + 0.5) * voxel_size
    zs = origin[2] + (np.arange(Z) + 0.5) * voxel_size
    step = max(1, (1 << 21) // (X * Y))
    for z0 in range(0, Z, step):
        z1 = min(Z, z0 + step)
        gz, gy, gx = np.meshgrid(zs[z0:z1], ys, xs, indexing="ij")
        p = np.stack([gx, gy, gz], axis=-1)
        out[z0:z1] = np.clip(scene_sdf(scene, p) / trunc, -1.0, 1.0).astype(np.float32)
    if half:
        out = out.astype(np.float16).astype(np.float32)
    tsdf = out.reshape(-1)
    weight = np.ones_like(tsdf)
    return tsdf, weight

"""Pinhole camera helpers and analytic ray casting (z-depth of the nearest hit along K^-1 (u,v,1)).

Camera frame: +z forward, +x right, +y down; pose = camera-to-world, row-major [R|t] (3x4).
Input generation only: nothing here is part of the method (section 3); depth maps are the
method's *input* (P:L81).
"""
from __future__ import annotations

import numpy as np

from .scene import Scene, scene_sdf


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(int(seed)))


def look_at(pos, target, up=(0.0, 0.0, 1.0)) -> np.ndarray:
    """Camera-to-world pose (3x4 float64) at `pos` looking at `target`."""
    pos = np.asarray(pos, dtype=np.float64)
    fwd = np.asarray(target, dtype=np.float64) - pos
    fwd /= np.linalg.norm(fwd)
    upv = np.asarray(up, dtype=np.float64)
    right = np.cross(fwd, upv)
    if np.linalg.norm(right) < 1e-6:
        right = np.cross(fwd, np.array([1.0, 0.0, 0.0]))
    right /= np.linalg.norm(right)
    down = np.cross(fwd, right)
    R = np.stack([right, down, fwd], axis=1)
    return np.concatenate([R, pos[:, None]], axis=1)


def rot_axis_angle(axis, angle_rad: float) -> np.ndarray:
    a = np.asarray(axis, dtype=np.float64)
    a = a / np.linalg.norm(a)
    Kx = np.array([[0, -a[2], a[1]], [a[2], 0, -a[0]], [-a[1], a[0], 0]])
    return np.eye(3) + np.sin(angle_rad) * Kx + (1 - np.cos(angle_rad)) * (Kx @ Kx)


def rotation_angle_deg(Ra: np.ndarray, Rb: np.ndarray) -> float:
    c = (np.trace(Ra.T @ Rb) - 1.0) * 0.5
    return float(np.degrees(np.arccos(np.clip(c, -1.0, 1.0))))


def compose_delta(pose: np.ndarray, axis, angle_rad: float, dtrans) -> np.ndarray:
    """Left-multiplied rotation about the camera centre plus a world-frame translation: the same
    pose family the method searches over (input perturbation only)."""
    R = rot_axis_angle(axis, angle_rad) @ pose[:, :3]
    t = pose[:, 3] + np.asarray(dtrans, dtype=np.float64)
    return np.concatenate([R, t[:, None]], axis=1)


def random_free_position(rng: np.random.Generator, scene: Scene, clearance: float) -> np.ndarray:
    for _ in range(4000):
        p = rng.uniform(scene.room_lo, scene.room_hi)
        if scene_sdf(scene, p) >= clearance:
            return p
    raise RuntimeError("no free position found")


def raycast_depth(scene: Scene, pose: np.ndarray, K, width: int, height: int) -> np.ndarray:
    """Exact z-depth image (float64, H x W) of the scene from camera-to-world `pose`.
    K = (fx, fy, cx, cy); pixel centres at integer (u, v)."""
    fx, fy, cx, cy = (float(v) for v in K)
    u = (np.arange(width, dtype=np.float64) - cx) / fx
    v = (np.arange(height, dtype=np.float64) - cy) / fy
    dc = np.stack(np.broadcast_arrays(u[None, :], v[:, None], np.ones((height, width))), axis=-1)
    R = np.asarray(pose[:, :3], dtype=np.float64)
    o = np.asarray(pose[:, 3], dtype=np.float64)
    d = dc @ R.T                                    # world direction with camera-z component 1
    with np.errstate(divide="ignore", invalid="ignore"):
        inv = 1.0 / d
        # room: we are inside; first exit through the slabs
        t_far = np.where(d > 0, (scene.room_hi - o) * inv, (scene.room_lo - o) * inv)
        t_far = np.where(d == 0, np.inf, t_far)
        best = np.min(t_far, axis=-1)
        for s in scene.spheres:
            oc = o - s[:3]
            a = np.sum(d * d, axis=-1)
            b = np.sum(d * oc, axis=-1)
            c = float(oc @ oc) - s[3] * s[3]
            disc = b * b - a * c
            sq = np.sqrt(np.maximum(disc, 0.0))
            t0 = (-b - sq) / a
            hit = (disc > 0) & (t0 > 1e-9)
            best = np.where(hit & (t0 < best), t0, best)
        for bx in scene.boxes:
            t1 = (bx[:3] - bx[3:] - o) * inv
            t2 = (bx[:3] + bx[3:] - o) * inv
            tn = np.max(np.minimum(t1, t2), axis=-1)
            tf = np.min(np.maximum(t1, t2), axis=-1)
            hit = (tn < tf) & (tn > 1e-9)
            best = np.where(hit & (tn < best), tn, best)
    return best          # camera-frame z because dc.z == 1


def add_noise(depth: np.ndarray, seed: int, sigma_abs: float = 0.0, sigma_rel: float = 0.0,
              dropout: float = 0.0) -> np.ndarray:
    """Gaussian depth noise (additive sigma_abs metres and/or multiplicative sigma_rel) and
    Bernoulli dropout to 0 (= invalid).  Returns float32."""
    rng = _rng(seed)
    z = depth.astype(np.float64)
    n = rng.standard_normal(z.shape)
    z = z + sigma_abs * n + sigma_rel * z * n
    if dropout > 0:
        z = np.where(rng.random(z.shape) < dropout, 0.0, z)
    return z.astype(np.float32)

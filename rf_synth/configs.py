"""The five BASELINE.json configs made concrete; all seeded, all synthetic.

Seeds: base = 210505600 + 1000*config; sub-streams +1 scene, +2 poses, +3 noise, +4 dropout,
+5/+6/+7 the three PSTs, +8 subsets.
"""
from __future__ import annotations

import numpy as np

from .camera import (add_noise, compose_delta, look_at, random_free_position, raycast_depth,
                     rot_axis_angle, rotation_angle_deg)
from .pst import sample_pst
from .scene import Scene, analytic_volume, make_scene, scene_sdf

BASE_SEED = 210505600

# (width, height, fx, fy, cx, cy) per config family
INTRINSICS = {
    1: (80, 60, 70.0, 70.0, 40.0, 30.0),
    2: (320, 240, 285.0, 285.0, 160.0, 120.0),
    3: (640, 480, 570.0, 570.0, 320.0, 240.0),
}


def config_seed(config: int, sub: int = 0) -> int:
    return BASE_SEED + 1000 * config + sub


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(int(seed)))


def _unit(rng: np.random.Generator) -> np.ndarray:
    v = rng.standard_normal(3)
    return v / np.linalg.norm(v)


# ----------------------------------------------------------------------------- config 1
def make_config1():
    """Tiny single-frame fitness: 64^3 fp32 analytic volume, one 80x60 frame, 1024 particles."""
    dims, vs, mu = (64, 64, 64), 0.02, 0.06
    scene = make_scene(config_seed(1, 1), extent=1.28, inset=mu + 2 * vs, n_spheres=3, n_boxes=0,
                       clearance=0.3)
    tsdf, weight = analytic_volume(scene, dims, vs, mu)
    rng = _rng(config_seed(1, 2))
    pos = None
    for clearance in (0.3, 0.25, 0.2, 0.15):          # the 1.08 m room is tight; documented fallback
        try:
            pos = random_free_position(rng, scene, clearance)
            break
        except RuntimeError:
            continue
    if pos is None:
        raise RuntimeError("config 1: no camera position")
    target = scene.spheres[int(rng.integers(len(scene.spheres))), :3]
    pose = look_at(pos, target)
    w, h, fx, fy, cx, cy = INTRINSICS[1]
    K = np.array([fx, fy, cx, cy], dtype=np.float32)
    depth = add_noise(raycast_depth(scene, pose, K, w, h), config_seed(1, 3), sigma_abs=0.002)
    pst = sample_pst(1024, config_seed(1, 5))
    return dict(dims=dims, voxel_size=vs, trunc=mu, scene=scene, tsdf=tsdf, weight=weight,
                pose=pose.astype(np.float32), K=K, width=w, height=h, depth=depth, pst=pst,
                scale=np.full(6, 0.05, dtype=np.float32))


# ----------------------------------------------------------------------------- config 2
def make_config2_inputs(n_build_frames: int = 30):
    """Tracking step: 256^3 fp32, room 2.56 m extent + 10 objects.  Returns the scene, the
    `n_build_frames` noisy frames + poses of a slow arc ending at T_prev (the volume is *built by
    integration* by whoever consumes this: the oracle in tests, the CUDA path in bench.py), the
    tracked frame rendered at T_true = Delta(15 deg, 8 cm) o T_prev, and three seeded PSTs."""
    dims, vs, mu = (256, 256, 256), 0.01, 0.04
    scene = make_scene(config_seed(2, 1), extent=2.56, inset=mu + 2 * vs, n_spheres=5, n_boxes=5,
                       clearance=0.3)
    w, h, fx, fy, cx, cy = INTRINSICS[2]
    K = np.array([fx, fy, cx, cy], dtype=np.float32)
    rng = _rng(config_seed(2, 2))
    centre = 0.5 * (scene.room_lo + scene.room_hi)
    # slow arc (about 1 cm and 0.3 deg per frame) at a seeded height, looking across the room
    for _ in range(1000):
        a0 = rng.uniform(0, 2 * np.pi)
        rad = rng.uniform(0.5, 0.8)
        zc = rng.uniform(centre[2] - 0.2, centre[2] + 0.2)
        angs = a0 + np.arange(n_build_frames) * (0.01 / rad)
        pos = np.stack([centre[0] + rad * np.cos(angs), centre[1] + rad * np.sin(angs),
                        np.full_like(angs, zc)], axis=1)
        if np.all(scene_sdf(scene, pos) >= 0.25):
            break
    else:
        raise RuntimeError("config 2: no clear arc")
    tgt = centre - 0.6 * (pos[n_build_frames // 2] - centre) + np.array([0, 0, -0.2])
    poses = [look_at(p, tgt) for p in pos]
    frames = [add_noise(raycast_depth(scene, T, K, w, h), config_seed(2, 3) + 17 * i, sigma_rel=0.01)
              for i, T in enumerate(poses)]
    T_prev = poses[-1]
    axis, direction = _unit(rng), _unit(rng)
    T_true = compose_delta(T_prev, axis, np.radians(15.0), 0.08 * direction)
    if scene_sdf(scene, T_true[:, 3]) < 0.15:
        T_true = compose_delta(T_prev, axis, np.radians(15.0), -0.08 * direction)
    tracked = add_noise(raycast_depth(scene, T_true, K, w, h), config_seed(2, 3) + 9999,
                        sigma_rel=0.01)
    psts = [sample_pst(n, config_seed(2, 5 + i)) for i, n in enumerate((1024, 3072, 10240))]
    return dict(dims=dims, voxel_size=vs, trunc=mu, scene=scene, K=K, width=w, height=h,
                build_poses=[T.astype(np.float32) for T in poses], build_frames=frames,
                T_prev=T_prev.astype(np.float32), T_true=T_true, tracked_depth=tracked, psts=psts,
                strides=(4, 8, 16))


# ----------------------------------------------------------------------------- configs 3, 4, 5
def make_config3_scene() -> Scene:
    """5.12 m extent, room 5.00 m, 12 objects (6 spheres + 6 boxes); shared by configs 3, 4, 5."""
    return make_scene(config_seed(3, 1), extent=5.12, inset=0.06, n_spheres=6, n_boxes=6,
                      clearance=0.4)


def _catmull_rom(P: np.ndarray, s: np.ndarray) -> np.ndarray:
    """Uniform Catmull-Rom through control points P (n,3) at parameters s in [1, n-2]."""
    i = np.clip(np.floor(s).astype(int), 1, len(P) - 3)
    t = (s - i)[:, None]
    p0, p1, p2, p3 = P[i - 1], P[i], P[i + 1], P[i + 2]
    return 0.5 * ((2 * p1) + (-p0 + p2) * t + (2 * p0 - 5 * p1 + 4 * p2 - p3) * t * t
                  + (-p0 + 3 * p1 - 3 * p2 + p3) * t * t * t)


def make_config3_trajectory(scene: Scene, n_frames: int = 200, step: float = 0.10,
                            max_rot_deg: float = 20.0, seed: int | None = None):
    """Camera-to-world poses (n_frames,3,4 float64): Catmull-Rom positions re-timed to a constant
    arclength `step` (0.10 m = 3 m/s at 30 fps, Table 1 L316-322 for the speed range) and
    look-at orientations towards a second, slower spline of targets; per-frame rotation clamped to
    `max_rot_deg`."""
    rng = _rng(config_seed(3, 2) if seed is None else seed)
    need = n_frames * step
    while True:
        keys = [random_free_position(rng, scene, 0.5) for _ in range(14)]
        P = np.array(keys)
        s = np.linspace(1.0, len(P) - 2.0, 20000)
        C = _catmull_rom(P, s)
        if np.any(scene_sdf(scene, C) < 0.3):
            continue
        seg = np.linalg.norm(np.diff(C, axis=0), axis=1)
        arc = np.concatenate([[0.0], np.cumsum(seg)])
        if arc[-1] >= need:
            break
    at = np.arange(n_frames) * step
    pos = np.stack([np.interp(at, arc, C[:, k]) for k in range(3)], axis=1)
    # targets: object centres visited in a seeded order, blended smoothly along the path
    objs = np.concatenate([scene.spheres[:, :3], scene.boxes[:, :3]], axis=0)
    order = rng.permutation(len(objs))
    tk = objs[np.concatenate([order, order[:3]])]
    ts = 1.0 + (at / need) * (len(tk) - 3.001)
    tgt = _catmull_rom(tk, ts)
    poses = np.zeros((n_frames, 3, 4))
    prev = None
    for i in range(n_frames):
        T = look_at(pos[i], tgt[i])
        if prev is not None:
            ang = rotation_angle_deg(prev[:, :3], T[:, :3])
            if ang > max_rot_deg:
                dR = T[:, :3] @ prev[:, :3].T
                ax = np.array([dR[2, 1] - dR[1, 2], dR[0, 2] - dR[2, 0], dR[1, 0] - dR[0, 1]])
                T[:, :3] = rot_axis_angle(ax, np.radians(max_rot_deg)) @ prev[:, :3]
        poses[i] = T
        prev = T
    return poses


def make_config5_poses(scene: Scene, n: int = 100) -> np.ndarray:
    """Random poses: position uniform with >= 0.5 m clearance, orientation uniform on SO(3)."""
    rng = _rng(config_seed(5, 2))
    out = np.zeros((n, 3, 4))
    for i in range(n):
        q = rng.standard_normal(4)
        q /= np.linalg.norm(q)
        w, x, y, z = q
        R = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                      [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                      [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])
        out[i, :, :3] = R
        out[i, :, 3] = random_free_position(rng, scene, 0.5)
    return out


def render_frame(scene: Scene, pose: np.ndarray, config: int, index: int, dropout: float = 0.05):
    """Noisy 640x480 frame of the config-3 scene (sigma = 1 % of depth, 5 % dropout)."""
    w, h, fx, fy, cx, cy = INTRINSICS[3]
    K = np.array([fx, fy, cx, cy], dtype=np.float32)
    d = raycast_depth(scene, pose, K, w, h)
    return add_noise(d, config_seed(config, 3) + 31 * index, sigma_rel=0.01, dropout=dropout), K

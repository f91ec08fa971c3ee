"""GPU parity of the surface point set (rf_extract_surface_points vs oracle O10): the same edges cross (bit-exact key
sets: integer work), every point within 1e-6 m of the oracle's (binary32 interpolation of exact sample values)."""
import numpy as np
import pytest

import oracle as orc
from test_gpu_parity import _rf, _small_world, _track_world

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _compare(vol, g, F, W):
    pts, edge = vol.extract_surface_points(cap=1 << 16)          # small first capacity: the re-call path is exercised
    pts, edge = pts.cpu().numpy(), edge.cpu().numpy()
    order = np.argsort(edge)
    pts, edge = pts[order], edge[order]
    want_p, want_e = orc.surface_points(g, F, W)
    assert np.array_equal(edge, want_e)
    assert np.max(np.abs(pts.astype(np.float64) - want_p)) <= 1e-6
    return len(want_e)


@pytest.mark.parametrize("dtype", [0, 1])
def test_surface_points_match_the_oracle(dtype):
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()          # 128^3, fused from 4 noisy frames
    if dtype == 1:
        F = F.astype(np.float16).astype(np.float32)
    vol = rf.Volume(dims, vs, mu, dtype=dtype)
    vol.upload(F, W)
    assert _compare(vol, g, F, W) > 5000
    vol.destroy()


def test_surface_points_ragged_volume_origin_and_empty():
    rf = _rf()
    dims, vs, mu = (70, 66, 50), 0.03, 0.09
    scene, K, w, h, poses, frames = _small_world(dims, vs, mu)
    origin = (0.4, -1.1, 2.3)
    g0 = orc.make_grid(dims, vs, mu)
    F, W = orc.empty_volume(dims)
    for T, d in zip(poses, frames):
        orc.integrate(g0, F, W, d, K, T, half_storage=True, nthreads=8)
    g = orc.make_grid(dims, vs, mu, origin)                     # the same samples on a grid that sits elsewhere
    vol = rf.Volume(dims, vs, mu, dtype=rf.RF_F16_W8, origin=origin)
    vol.upload(F, W)
    assert _compare(vol, g, F, W) > 500
    vol.reset()
    pts, edge = vol.extract_surface_points()
    assert pts.shape[0] == 0 and edge.shape[0] == 0
    vol.destroy()

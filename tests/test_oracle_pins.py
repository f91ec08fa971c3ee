"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests re-types the oracle's formula and compares it with itself: each pin is a closed
form, an invariant, a library routine (scipy) or a brute-force loop written independently here.
"""
import math
import os

import numpy as np
import pytest
from scipy import ndimage
from scipy.spatial.transform import Rotation

import oracle as orc
import rf_synth as S

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")


def _gold():
    out = {}
    for line in open(GOLD):
        line = line.split("#")[0].split()
        if line:
            out[line[0]] = [float(v) for v in line[1:]]
    return out


# ---------------------------------------------------------------------------------- constants
def test_paper_constants():
    g = _gold()
    assert orc.const(orc.TAU) == g["tau"][0]
    assert orc.const(orc.EPS) == g["epsilon"][0]
    assert orc.const(orc.BETA) == g["beta"][0]
    assert orc.const(orc.STOP_TOL) == g["stop_tol"][0]
    assert orc.const(orc.EMPTY_STOP) == g["empty_stop"][0]


# ---------------------------------------------------------------------------------- P1  PST
@pytest.mark.parametrize("n,seed", [(1024, 11), (10240, 12)])
def test_p1_pst_uniform_in_unit_6_ball(n, seed):
    p = S.sample_pst(n, seed).astype(np.float64)
    r = np.linalg.norm(p, axis=1)
    assert p.shape == (n, 6) and np.all(r <= 1.0)
    # radial CDF is r^6 (uniform 6-ball): Kolmogorov-Smirnov at the 5 % level
    u = np.sort(r ** 6)
    d = max(np.max(np.arange(1, n + 1) / n - u), np.max(u - np.arange(n) / n))
    assert d < 1.358 / math.sqrt(n)
    # closed-form moments of the uniform d-ball, d = 6
    assert abs(r.mean() - 6 / 7) < 4 * math.sqrt((6 / 8 - (6 / 7) ** 2) / n)
    frac = np.mean(r < 0.5)
    assert abs(frac - 1 / 64) < 4 * math.sqrt((1 / 64) * (63 / 64) / n)
    cov = p.T @ p / n
    assert np.all(np.abs(p.mean(axis=0)) < 4 * math.sqrt(1 / 8 / n))
    # Var(x_i) = 1/(d+2) = 1/8 ; Var(x_i^2) = 3/((d+2)(d+4)) - 1/64 ; Var(x_i x_j) = 1/((d+2)(d+4))
    assert np.all(np.abs(np.diag(cov) - 1 / 8) < 4 * math.sqrt((3 / 80 - 1 / 64) / n))
    off = cov - np.diag(np.diag(cov))
    assert np.all(np.abs(off) < 4.5 * math.sqrt((1 / 80) / n))


def test_p1_pst_seeded_and_distinct():
    a, b, c = S.sample_pst(256, 5), S.sample_pst(256, 5), S.sample_pst(256, 6)
    assert np.array_equal(a, b) and not np.array_equal(a, c) and a.dtype == np.float32


def test_p1_poisson_disk_pst():
    """SURVEY 8(f)-2 / P:L284: 6-D Poisson-disk template.  Every particle inside the unit ball, no two closer than the
    returned radius, seeded; nearest-neighbour distances have a hard floor well above the i.i.d. template's."""
    from scipy.spatial import cKDTree
    n = 1024
    p, r = S.sample_pst_poisson(n, 31, return_radius=True)
    assert p.shape == (n, 6) and p.dtype == np.float32
    assert np.all(np.linalg.norm(p.astype(np.float64), axis=1) <= 1.0)
    nn = cKDTree(p.astype(np.float64)).query(p.astype(np.float64), k=2)[0][:, 1]
    assert nn.min() >= r * (1 - 1e-5) and r > 0.3
    q = S.sample_pst(n, 31)
    nn_iid = cKDTree(q.astype(np.float64)).query(q.astype(np.float64), k=2)[0][:, 1]
    assert nn.min() > 2.0 * nn_iid.min()
    assert np.array_equal(p, S.sample_pst_poisson(n, 31)) and not np.array_equal(p, S.sample_pst_poisson(n, 32))
    # still an unbiased cover of the ball: mean near 0, radial mass concentrated near the surface like r^6
    assert np.all(np.abs(p.mean(0)) < 0.05) and 0.75 < np.linalg.norm(p, axis=1).mean() < 0.92


# ---------------------------------------------------------------------------------- P2  pose algebra
def test_p2_identity_and_orthonormal():
    rng = np.random.default_rng(0)
    T = np.concatenate([Rotation.random(random_state=1).as_matrix(), rng.normal(size=(3, 1))], axis=1)
    assert np.allclose(orc.apply_delta(T, np.zeros(6)), T, atol=0, rtol=0)
    for _ in range(50):
        d = rng.uniform(-1, 1, 6)
        d[:3] *= rng.uniform(0, 1) / max(1e-9, np.linalg.norm(d[:3]))
        Tn = orc.apply_delta(T, d)
        Rn = Tn[:, :3]
        assert np.allclose(Rn.T @ Rn, np.eye(3), atol=1e-12)
        assert abs(np.linalg.det(Rn) - 1) < 1e-12
        # rotation angle of the increment = 2 asin |delta_q|  (unit quaternion with imaginary part delta_q)
        dR = Rn @ T[:, :3].T
        ang = math.acos(np.clip((np.trace(dR) - 1) / 2, -1, 1))
        assert abs(ang - 2 * math.asin(np.linalg.norm(d[:3]))) < 1e-7
        # translation increment is a plain world-frame addition
        assert np.allclose(Tn[:, 3], T[:, 3] + d[3:], atol=1e-15)


def test_p2_textbook_x_rotation_and_scipy():
    th = 0.7
    I = np.concatenate([np.eye(3), np.zeros((3, 1))], axis=1)
    Tn = orc.apply_delta(I, [math.sin(th / 2), 0, 0, 0, 0, 0])
    Rx = np.array([[1, 0, 0], [0, math.cos(th), -math.sin(th)], [0, math.sin(th), math.cos(th)]])
    assert np.allclose(Tn[:, :3], Rx, atol=1e-15)
    rng = np.random.default_rng(3)
    for _ in range(20):
        q = rng.normal(size=4)
        q /= np.linalg.norm(q)
        assert np.allclose(orc.quat_to_R(q), Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix(), atol=1e-14)


def test_p2_left_multiplication_and_inverse():
    # Delta(d) o T then Delta(-d) o (.) returns T (same |d_q| -> conjugate quaternion)
    rng = np.random.default_rng(4)
    T = np.concatenate([Rotation.random(random_state=2).as_matrix(), rng.normal(size=(3, 1))], axis=1)
    d = np.array([0.1, -0.2, 0.05, 0.3, -0.1, 0.2])
    back = orc.apply_delta(orc.apply_delta(T, d), -d)
    assert np.allclose(back, T, atol=1e-14)
    # the increment is applied on the LEFT of R_c (world-frame axis), reading A2
    Rq = Rotation.from_quat([d[0], d[1], d[2], math.sqrt(1 - d[:3] @ d[:3])]).as_matrix()
    assert np.allclose(orc.apply_delta(T, d)[:, :3], Rq @ T[:, :3], atol=1e-14)
    # pose_from_particle = apply_delta with delta = r (.) p
    p = np.array([0.3, -0.1, 0.2, 0.5, 0.1, -0.4], dtype=np.float32)
    r = np.array([0.05, 0.02, 0.03, 0.1, 0.2, 0.05])
    assert np.allclose(orc.pose_from_particle(T, r, p), orc.apply_delta(T, r * p.astype(np.float64)), atol=1e-15)


# ---------------------------------------------------------------------------------- P3  back-projection
def test_p3_backprojection():
    w, h = 64, 48
    K = np.array([50.0, 55.0, 32.0, 24.0], dtype=np.float32)
    rng = np.random.default_rng(5)
    depth = rng.uniform(0.5, 3.0, (h, w)).astype(np.float32)
    depth[10, 20] = 0.0
    depth[11, 21] = np.nan
    depth[12, 22] = -1.0
    pts = orc.backproject(depth, K, 1)
    assert pts.shape == (w * h, 4)
    c = pts[24 * w + 32]
    assert c[0] == 0 and c[1] == 0 and c[2] == depth[24, 32] and c[3] == 1
    for (v, u) in [(10, 20), (11, 21), (12, 22)]:
        assert pts[v * w + u, 3] == 0
    # project o back-project = identity on the lattice
    ok = pts[:, 3] == 1
    uu = K[0] * pts[ok, 0] / pts[ok, 2] + K[2]
    vv = K[1] * pts[ok, 1] / pts[ok, 2] + K[3]
    U, V = np.meshgrid(np.arange(w), np.arange(h))
    assert np.allclose(uu, U.reshape(-1)[ok], atol=1e-9) and np.allclose(vv, V.reshape(-1)[ok], atol=1e-9)
    # stride lattice: (W/s)(H/s) samples at phase floor(s/2)
    for s in (2, 4, 8, 16):
        ps = orc.backproject(depth, K, s)
        assert ps.shape[0] == (w // s) * (h // s)
        first = ps[0]
        assert first[2] == depth[s // 2, s // 2]
    assert orc.lattice_count(640, 8) == 80 and orc.lattice_count(480, 32) == 15 and orc.lattice_count(3, 8) == 0


# ---------------------------------------------------------------------------------- P4  integration
def _grid(n=32, vs=0.05, mu=0.15, origin=(-0.8, -0.8, 0.0)):
    return orc.make_grid((n, n, n), vs, mu, origin), n, vs, mu, np.array(origin)


def _centres(n, vs, origin):
    c = origin[None, :] + (np.stack(np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij"), -1)
                           .reshape(-1, 3) + 0.5) * vs          # order i,j,k with k fastest
    lin = (np.arange(n)[:, None, None] + n * (np.arange(n)[None, :, None] + n * np.arange(n)[None, None, :])).reshape(-1)
    out = np.zeros((n ** 3, 3))
    out[lin] = c
    return out       # indexed by x + X*(y + Y*z)


IDENT = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0]], dtype=np.float32)


def test_p4_plane_closed_form():
    g, n, vs, mu, org = _grid()
    w, h = 64, 48
    K = np.array([40.0, 40.0, 31.5, 23.5], dtype=np.float32)
    d0 = 1.0
    depth = np.full((h, w), d0, dtype=np.float32)
    F, W = orc.empty_volume((n, n, n))
    orc.integrate(g, F, W, depth, K, IDENT)
    c = _centres(n, vs, org)
    z = c[:, 2]
    u = K[0] * c[:, 0] / z + K[2]
    v = K[1] * c[:, 1] / z + K[3]
    inimg = (np.floor(u + 0.5) >= 0) & (np.floor(u + 0.5) < w) & (np.floor(v + 0.5) >= 0) & (np.floor(v + 0.5) < h)
    upd = inimg & (d0 - z >= -mu)
    # voxels whose decision sits within rounding of a boundary are left out of the pin
    safe = (np.abs((u + 0.5) - np.round(u + 0.5)) > 1e-3) & (np.abs((v + 0.5) - np.round(v + 0.5)) > 1e-3) \
        & (np.abs(d0 - z + mu) > 1e-5)
    expect = np.minimum(1.0, (d0 - z) / mu)     # exact truncated signed distance to the plane z = d0
    assert np.all(W[upd & safe] == 1) and np.all(W[~upd & safe] == 0)
    assert np.allclose(F[upd & safe], expect[upd & safe], atol=2e-6)
    assert np.all(F[~upd & safe] == 1.0)
    assert upd.sum() > 5000 and (expect[upd] < 0).sum() > 500


def test_p4_sphere_closed_form():
    g, n, vs, mu, org = _grid()
    w, h = 64, 48
    K = np.array([40.0, 40.0, 31.5, 23.5], dtype=np.float64)
    rs = 1.2
    U, V = np.meshgrid(np.arange(w), np.arange(h))
    ray = np.stack([(U - K[2]) / K[0], (V - K[3]) / K[1], np.ones_like(U, dtype=np.float64)], -1)
    depth = (rs / np.linalg.norm(ray, axis=-1)).astype(np.float32)      # z-depth of a sphere centred on the camera
    F, W = orc.empty_volume((n, n, n))
    orc.integrate(g, F, W, depth, K.astype(np.float32), IDENT)
    c = _centres(n, vs, org)
    z = c[:, 2]
    uf, vf = K[0] * c[:, 0] / z + K[2], K[1] * c[:, 1] / z + K[3]
    ur, vr = np.floor(uf + 0.5).astype(int), np.floor(vf + 0.5).astype(int)
    inimg = (ur >= 0) & (ur < w) & (vr >= 0) & (vr < h)
    safe = (np.abs((uf + 0.5) - np.round(uf + 0.5)) > 1e-3) & (np.abs((vf + 0.5) - np.round(vf + 0.5)) > 1e-3)
    d = np.where(inimg, depth[np.clip(vr, 0, h - 1), np.clip(ur, 0, w - 1)].astype(np.float64), np.nan)
    sdf = d - z
    safe &= np.abs(sdf + mu) > 1e-5
    upd = inimg & (sdf >= -mu)
    expect = np.minimum(1.0, sdf / mu)
    assert np.allclose(F[upd & safe], expect[upd & safe], atol=2e-6)
    assert np.all(W[upd & safe] == 1) and np.all(W[~upd & safe] == 0)
    # projective sdf = (true distance to the sphere) * cos(theta) up to the pixel quantisation:
    near = upd & safe & (np.abs(sdf) < mu)
    true_dist = rs - np.linalg.norm(c, axis=1)
    cos = z / np.linalg.norm(c, axis=1)
    assert np.max(np.abs(sdf[near] - true_dist[near] * cos[near])) < 0.03


def _plane_view(origin, rotvec, t, w=64, h=48, n=32, vs=0.05, mu=0.15):
    """A world plane n.x = c seen from the camera [R|t] (camera-to-world): closed-form depth image
    D(u,v) = (c - n.t) / (n . R K^-1 (u,v,1))  (the z-depth at which the pixel ray t + R K^-1(u,v,1) D meets the plane)."""
    g = orc.make_grid((n, n, n), vs, mu, origin)
    K = np.array([44.0, 41.0, 30.7, 24.2])
    R = Rotation.from_rotvec(rotvec).as_matrix()
    t = np.asarray(t, dtype=np.float64)
    nrm = R @ np.array([0.25, -0.2, 1.0])            # roughly facing the camera, tilted
    nrm /= np.linalg.norm(nrm)
    c = nrm @ (t + R @ np.array([0.0, 0.0, 1.1]))    # the optical axis meets the plane at depth 1.1
    U, V = np.meshgrid(np.arange(w), np.arange(h))
    ray = np.stack([(U - K[2]) / K[0], (V - K[3]) / K[1], np.ones_like(U, dtype=np.float64)], -1)
    den = (ray @ R.T) @ nrm
    D = (c - nrm @ t) / den
    depth = np.where((den > 0) & (D > 0), D, 0.0).astype(np.float32)
    pose = np.concatenate([R, t[:, None]], 1).astype(np.float32)
    return g, K.astype(np.float32), pose, depth, nrm, c


@pytest.mark.parametrize("origin,rotvec,t", [
    ((-0.8, -0.8, 0.0), (0.0, 0.0, 0.0), (0.0, 0.0, 0.0)),                      # the identity, as a control
    ((-0.6, -0.9, 0.1), (0.3, -0.5, 0.2), (0.25, -0.1, -0.05)),                 # rotated and translated camera, origin != 0
    ((0.4, 0.3, -0.2), (-0.4, 0.7, -1.1), (0.9, 1.5, 0.1)),                     # a large rotation (about 80 deg), camera off-grid
])
def test_p4_plane_from_a_rotated_translated_camera(origin, rotvec, t):
    """Pins the pose handling of O9 (R^T, not R; p_w - t, not p_w + t; row/column order; origin; the +1/2 cell centre):
    the expected values come from an independent numpy evaluation and, separately, from the ray-plane intersection of
    each voxel's OWN viewing ray (no pixel logic at all), which the projective sdf must match up to pixel quantisation."""
    n, vs, mu, w, h = 32, 0.05, 0.15, 64, 48
    g, K, pose, depth, nrm, c = _plane_view(origin, rotvec, t, w, h, n, vs, mu)
    F, W = orc.empty_volume((n, n, n))
    frag = np.zeros(n ** 3, dtype=np.uint8)
    orc.integrate(g, F, W, depth, K, pose, fragile=frag)
    R, tt = pose[:, :3].astype(np.float64), pose[:, 3].astype(np.float64)
    P = _centres(n, vs, np.array(origin))
    pc = (P - tt) @ R                                # row-vector form of R^T (p - t)
    z = pc[:, 2]
    front = z > 1e-9
    zs = np.where(front, z, 1.0)
    uf, vf = K[0] * pc[:, 0] / zs + K[2], K[1] * pc[:, 1] / zs + K[3]
    ur, vr = np.floor(uf + 0.5).astype(int), np.floor(vf + 0.5).astype(int)
    inimg = front & (ur >= 0) & (ur < w) & (vr >= 0) & (vr < h)
    d = np.where(inimg, depth[np.clip(vr, 0, h - 1), np.clip(ur, 0, w - 1)].astype(np.float64), 0.0)
    sdf = d - z
    upd = inimg & (d > 0) & (sdf >= -mu)
    safe = (np.abs((uf + 0.5) - np.round(uf + 0.5)) > 1e-3) & (np.abs((vf + 0.5) - np.round(vf + 0.5)) > 1e-3) \
        & (np.abs(sdf + mu) > 1e-5) & (np.abs(z) > 1e-5)
    assert np.all(W[upd & safe] == 1) and np.all(W[~upd & safe] == 0)
    assert np.allclose(F[upd & safe], np.minimum(1.0, sdf[upd & safe] / mu), atol=1e-6)
    assert np.all(F[~upd & safe] == 1.0)
    assert upd.sum() > 3000 and (sdf[upd] < 0).sum() > 200 and (W == 0).sum() > 3000
    # the oracle's own fragile flags (R-I2) mark only voxels that this independent evaluation also finds near a boundary
    assert not np.any(safe & (frag == 1)) and frag.mean() < 0.01
    # geometry only: along the voxel's own ray the plane lies at z * (c - n.t) / (n.(p - t)); the image stores that depth at
    # the nearest pixel centre, so the two differ by at most half a pixel of depth slope in u plus half a pixel in v
    near = upd & safe & (np.abs(sdf) < mu) & (ur >= 1) & (ur < w - 1) & (vr >= 1) & (vr < h - 1)
    s = (c - nrm @ tt) / ((P - tt) @ nrm)
    own = z * s - z
    D = depth.astype(np.float64)
    slope = 0.5 * (np.abs(D[vr[near], ur[near] + 1] - D[vr[near], ur[near] - 1]) + np.abs(D[vr[near] + 1, ur[near]] - D[vr[near] - 1, ur[near]]))
    assert near.sum() > 1000
    assert np.all(np.abs(sdf[near] - own[near]) <= 0.55 * slope + 1e-6)
    assert np.all(np.abs(F[near] - own[near] / mu) <= (0.55 * slope + 1e-6) / mu + 1e-6)


def test_p4_fragile_flags_mark_exactly_the_near_boundary_voxels():
    """R-I2: a voxel is flagged iff a move of p_c by eps_p = 2e-6 m can change its pixel, its z > 0 test or its band test.
    Constructed cases: a camera whose optical axis passes exactly through a row of voxel centres (u = cx exactly: not
    fragile) and one shifted by half a pixel footprint (u = cx + 1/2: a rounding boundary, fragile)."""
    n, vs, mu = 16, 0.125, 0.375                       # binary-exact geometry
    g = orc.make_grid((n, n, n), vs, mu, (0.0, 0.0, 0.0))
    w, h = 33, 33
    eps = orc.integrate_eps_p()
    assert eps == 2e-6
    depth = np.full((h, w), 1.5, dtype=np.float32)
    lin = lambda i, j, k: i + n * (j + n * k)
    col = [lin(8, 8, k) for k in range(n)]           # voxel centres (1.0625, 1.0625, (k+1/2)/8)
    for shift, expect in ((0.0, 0), (0.5, 1)):
        # fx chosen so that one pixel spans 1/64 m at depth z = 1: x_c = shift/64 at z = 1 projects to cx + shift
        K = np.array([64.0, 64.0, 16.0, 16.0], dtype=np.float32)
        pose = np.array([[1, 0, 0, 1.0625 - shift / 64.0], [0, 1, 0, 1.0625], [0, 0, 1, -0.9375 + 0.0]], dtype=np.float32)
        F, W = orc.empty_volume((n, n, n))
        frag = np.zeros(n ** 3, dtype=np.uint8)
        orc.integrate(g, F, W, depth, K, pose, fragile=frag)
        k1 = 0                                        # voxel (8,8,0): z = 0.0625 + 0.9375 = 1.0 exactly
        assert frag[col[k1]] == expect, (shift, frag[col[k1]])
    # band test: a voxel exactly mu behind the surface is fragile, one 1e-4 m off is not
    K = np.array([64.0, 64.0, 16.0, 16.0], dtype=np.float32)
    pose = np.array([[1, 0, 0, 1.0625], [0, 1, 0, 1.0625], [0, 0, 1, -0.9375]], dtype=np.float32)
    for d0, expect in ((1.0 - 0.375, 1), (1.0 - 0.375 + 1e-4, 0), (1.0 - 0.375 - 1e-4, 0)):
        F, W = orc.empty_volume((n, n, n))
        frag = np.zeros(n ** 3, dtype=np.uint8)
        orc.integrate(g, F, W, np.full((h, w), d0, dtype=np.float32), K, pose, fragile=frag)
        assert frag[col[0]] == expect, d0
        assert W[col[0]] == (1 if d0 >= 1.0 - 0.375 else 0)
    # z > 0 test: a camera whose z = 0 plane passes through a layer of voxel centres
    pose0 = np.array([[1, 0, 0, 1.0625], [0, 1, 0, 1.0625], [0, 0, 1, 0.0625]], dtype=np.float32)
    frag = np.zeros(n ** 3, dtype=np.uint8)
    F, W = orc.empty_volume((n, n, n))
    orc.integrate(g, F, W, depth, K, pose0, fragile=frag)
    layer0 = np.array([lin(i, j, 0) for i in range(n) for j in range(n)])
    assert np.all(frag[layer0] == 1) and np.all(W[layer0] == 0)


def test_p4_running_average_and_cap():
    g, n, vs, mu, org = _grid(n=16, vs=0.1, mu=0.3, origin=(-0.8, -0.8, 0.0))
    w, h = 32, 24
    K = np.array([20.0, 20.0, 15.5, 11.5], dtype=np.float32)
    F, W = orc.empty_volume((n, n, n))
    d1, d2 = 1.0, 1.1
    orc.integrate(g, F, W, np.full((h, w), d1, np.float32), K, IDENT)
    F1 = F.copy()
    orc.integrate(g, F, W, np.full((h, w), d2, np.float32), K, IDENT)
    c = _centres(n, vs, org)
    z = c[:, 2]
    both = (W == 2)
    e = 0.5 * (np.minimum(1, (d1 - z) / mu) + np.minimum(1, (np.float32(d2) - z) / mu))
    assert both.sum() > 300 and np.allclose(F[both], e[both], atol=2e-6)
    only2 = (W == 1) & (F1 == 1.0) & (F != 1.0)
    assert only2.sum() > 0      # band of the second plane only
    # n identical frames -> same F, W = min(n, w_max); beyond the cap an EMA with factor w_max/(w_max+1)
    F, W = orc.empty_volume((n, n, n))
    for _ in range(5):
        orc.integrate(g, F, W, np.full((h, w), d1, np.float32), K, IDENT, w_max=3)
    seen = W > 0
    assert np.all(W[seen] == 3) and np.allclose(F[seen], np.minimum(1, (d1 - z[seen]) / mu), atol=2e-6)
    Fb = F.copy()
    orc.integrate(g, F, W, np.full((h, w), d2, np.float32), K, IDENT, w_max=3)
    both = seen & (np.float32(d2) - z >= -mu)
    e = (3 * Fb[both] + np.minimum(1, (np.float32(d2) - z[both]) / mu)) / 4
    assert np.allclose(F[both], e, atol=2e-6) and np.all(W[both] == 3)


def test_p4_half_storage_rounding_matches_numpy_float16():
    rng = np.random.default_rng(7)
    v = np.concatenate([rng.uniform(-1, 1, 4000), rng.uniform(-1e-4, 1e-4, 500), rng.uniform(-7e-8, 7e-8, 200),
                        [0.0, 1.0, -1.0, 0.5, 2 ** -14, 2 ** -24, 1.5 * 2 ** -24, 0.99951171875, 0.999755859375]])
    ours = np.array([orc.round_to_half(x) for x in v])
    ref = v.astype(np.float16).astype(np.float64)           # numpy rounds binary64 -> binary16 with RNE
    assert np.array_equal(ours, ref)


def test_p4_subset_equals_full():
    g, n, vs, mu, org = _grid()
    w, h = 64, 48
    K = np.array([40.0, 40.0, 31.5, 23.5], dtype=np.float32)
    rng = np.random.default_rng(8)
    depth = rng.uniform(0.6, 1.4, (h, w)).astype(np.float32)
    pose = S.look_at([0.1, -0.05, 0.0], [0.0, 0.1, 1.0], up=(0, -1, 0)).astype(np.float32)
    F, W = orc.empty_volume((n, n, n))
    lin = rng.choice(n ** 3, 3000, replace=False)
    Fs, Ws = F[lin].copy(), W[lin].copy()
    for _ in range(2):
        orc.integrate(g, F, W, depth, K, pose, half_storage=True)
        orc.integrate_subset(g, lin, Fs, Ws, depth, K, pose, half_storage=True)
    assert np.array_equal(F[lin], Fs) and np.array_equal(W[lin], Ws) and (W > 0).sum() > 1000


# ---------------------------------------------------------------------------------- P5  trilinear
def test_p5_affine_reproduction_and_bounds():
    n, vs = 12, 0.125                    # exactly representable in binary32, so centres are exact
    org = np.array([0.25, -0.5, 1.0])
    g = orc.make_grid((n, n + 2, n + 4), vs, 0.375, org)
    X, Y, Z = n, n + 2, n + 4
    a = np.array([0.31, -0.17, 0.23])
    d = 0.05
    ii, jj, kk = np.meshgrid(np.arange(X), np.arange(Y), np.arange(Z), indexing="ij")
    cen = org + (np.stack([ii, jj, kk], -1) + 0.5) * vs
    field = np.zeros(X * Y * Z, dtype=np.float32)
    lin = (ii + X * (jj + Y * kk)).reshape(-1)
    vals = (cen.reshape(-1, 3) @ a + d)
    field[lin] = vals.astype(np.float32)
    Wt = np.ones_like(field)
    rng = np.random.default_rng(9)
    lo = org + 0.5 * vs
    hi = org + (np.array([X, Y, Z]) - 0.5) * vs
    for _ in range(300):
        p = rng.uniform(lo, hi - 1e-9)
        ok, psi, _ = orc.trilinear(g, field, Wt, p)
        assert ok and abs(psi - (p @ a + d)) < 2e-7          # float32 storage of the field
    # voxel centres return the voxel value; index order x fastest
    for (i, j, k) in [(0, 0, 0), (3, 5, 7), (X - 2, Y - 2, Z - 2)]:
        ok, psi, _ = orc.trilinear(g, field, Wt, org + (np.array([i, j, k]) + 0.5) * vs)
        assert ok and psi == pytest.approx(float(field[i + X * (j + Y * k)]), abs=1e-7)
    # half-open bound rule: g = dim-1 (last voxel centre) is outside, just below is inside
    last = org + (np.array([X - 1, 3, 3]) + 0.5) * vs
    assert not orc.trilinear(g, field, Wt, last)[0]
    assert orc.trilinear(g, field, Wt, last - np.array([1e-6, 0, 0]))[0]
    assert not orc.trilinear(g, field, Wt, org + np.array([0.49, 3, 3]) * vs)[0]      # g < 0
    # an unobserved corner invalidates the whole cell, even with zero interpolation weight
    W2 = Wt.copy()
    W2[4 + X * (4 + Y * 4)] = 0
    assert not orc.trilinear(g, field, W2, org + (np.array([3.5, 3.5, 3.5]) + 0.5) * vs)[0]
    assert not orc.trilinear(g, field, W2, org + (np.array([3.0, 3.0, 3.0]) + 0.5) * vs)[0]
    assert orc.trilinear(g, field, W2, org + (np.array([2.5, 3.5, 3.5]) + 0.5) * vs)[0]


def test_p5_scipy_map_coordinates():
    X, Y, Z = 9, 10, 11
    rng = np.random.default_rng(10)
    vol = rng.uniform(-1, 1, (Z, Y, X)).astype(np.float32)
    vs = 0.03125                                   # exactly representable in binary32
    g = orc.make_grid((X, Y, Z), vs, 0.09375, (0.125, 0.25, 0.5))
    field = vol.reshape(-1)
    Wt = np.ones_like(field)
    org = np.array([0.125, 0.25, 0.5])
    gc = rng.uniform(0, [X - 1.001, Y - 1.001, Z - 1.001], (200, 3))
    ref = ndimage.map_coordinates(vol.astype(np.float64), [gc[:, 2], gc[:, 1], gc[:, 0]], order=1)
    for q, r in zip(gc, ref):
        ok, psi, _ = orc.trilinear(g, field, Wt, org + (q + 0.5) * vs)
        assert ok and abs(psi - r) < 1e-9


# ---------------------------------------------------------------------------------- P6  fitness
def _plane_setup():
    """Plane z = d0 integrated once at identity; noise-free points on that plane."""
    n, vs, mu = 48, 0.05, 0.15
    org = np.array([-1.2, -1.2, 0.0])
    g = orc.make_grid((n, n, n), vs, mu, org)
    w, h = 64, 48
    K = np.array([60.0, 60.0, 31.5, 23.5], dtype=np.float32)
    d0 = 1.5
    depth = np.full((h, w), d0, dtype=np.float32)
    F, W = orc.empty_volume((n, n, n))
    orc.integrate(g, F, W, depth, K, IDENT)
    pts = orc.backproject(depth, K, 2).astype(np.float32)
    # keep interior points: cells at the image border touch voxels the frame never observed
    pts = np.ascontiguousarray(pts[(np.abs(pts[:, 0]) < 0.55) & (np.abs(pts[:, 1]) < 0.40)])
    return g, F, W, pts, mu, vs


def test_p6_plane_translation_closed_form():
    g, F, W, pts, mu, vs = _plane_setup()
    M = pts.shape[0]
    zero = np.zeros((1, 6), dtype=np.float32)
    one = np.ones(6, dtype=np.float32)
    r = orc.eval_particles(g, F, W, pts, zero, IDENT, one)
    assert r["M_O"] == M and r["n"][0] == M and r["S"][0] < 1e-10 and abs(r["rho"][0] - 1) < 1e-10
    prev = 1.0
    for a in (0.02, 0.05, -0.05, 0.10, -0.12):
        # camera moved by +a along z: every point sits a beyond the plane -> psi = -a/mu for all points
        pst = np.array([[0, 0, 0, 0, 0, a]], dtype=np.float32)
        r = orc.eval_particles(g, F, W, pts, pst, IDENT, one)
        assert r["n"][0] == M
        assert r["S"][0] == pytest.approx(M * (a / mu) ** 2, rel=1e-5)
        assert r["rho"][0] == pytest.approx(math.exp(-(a / mu) ** 2), rel=1e-5)      # pins tau, square, 1/|O|, units
        # sign: psi is negative behind the surface (a > 0)
        ok, psi, _ = orc.trilinear(g, F, W, pts[M // 2, :3].astype(np.float64) + np.array([0, 0, a]))
        assert ok and psi == pytest.approx(-a / mu, abs=1e-5)
    for a in (0.01, 0.03, 0.06, 0.09, 0.12):           # monotone in |a|
        pst = np.array([[0, 0, 0, 0, 0, a]], dtype=np.float32)
        cur = orc.eval_particles(g, F, W, pts, pst, IDENT, one)["rho"][0]
        assert cur < prev
        prev = cur
    # in-plane translation leaves the fitness unchanged while all points stay observed
    pst = np.array([[0, 0, 0, 0.07, -0.04, 0]], dtype=np.float32)
    r = orc.eval_particles(g, F, W, pts, pst, IDENT, one)
    assert r["n"][0] == M and r["rho"][0] == pytest.approx(1.0, abs=1e-9)


def test_p6_points_leaving_the_grid_count_and_F2():
    g, F, W, pts, mu, vs = _plane_setup()
    M = pts.shape[0]
    one = np.ones(6, dtype=np.float32)
    shift = 0.9
    pst = np.array([[0, 0, 0, shift, 0, 0]], dtype=np.float32)
    r = orc.eval_particles(g, F, W, pts, pst, IDENT, one)
    # a point is sampleable iff its 2x2x2 cell is inside the grid and all corners were observed by the
    # identity-pose frame; count geometrically with an independent check of the weights
    X = 48
    gx = (pts[:, 0].astype(np.float64) + shift + 1.2) / vs - 0.5
    gy = (pts[:, 1].astype(np.float64) + 1.2) / vs - 0.5
    gz = (pts[:, 2].astype(np.float64)) / vs - 0.5
    Wv = W.reshape(48, 48, 48)      # [z,y,x]
    cnt = 0
    for x, y, z in zip(gx, gy, gz):
        i, j, k = int(math.floor(x)), int(math.floor(y)), int(math.floor(z))
        if 0 <= i and i + 1 <= X - 1 and 0 <= j and j + 1 <= X - 1 and 0 <= k and k + 1 <= X - 1:
            if np.all(Wv[k:k + 2, j:j + 2, i:i + 2] > 0):
                cnt += 1
    assert 0 < cnt < M and r["n"][0] == cnt
    assert r["rho"][0] == pytest.approx(math.exp(-(r["S"][0] + (M - cnt)) / M), rel=1e-12)     # F2 (A6)
    f1 = orc.eval_particles(g, F, W, pts, pst, IDENT, one, mode=1)
    exp_f1 = 0.0 if cnt < M / 2 else math.exp(-r["S"][0] / cnt)
    assert f1["rho"][0] == pytest.approx(exp_f1, rel=1e-12)
    # masked points are skipped and do not count in M_O
    p2 = pts.copy()
    p2[::3, 3] = 0
    r2 = orc.eval_particles(g, F, W, p2, np.zeros((1, 6), np.float32), IDENT, one)
    assert r2["M_O"] == M - len(p2[::3]) and r2["n"][0] == r2["M_O"]


def test_p6_brute_force_16cube():
    """Independent literal 8-corner loop on a random 16^3 grid (north_star)."""
    n, vs, mu = 16, 0.04, 0.12
    org = np.array([0.05, -0.1, 0.2], dtype=np.float32).astype(np.float64)    # the grid stores binary32
    rng = np.random.default_rng(12)
    vol = rng.uniform(-1, 1, (n, n, n)).astype(np.float32)      # [z,y,x]
    wgt = (rng.random((n, n, n)) > 0.03).astype(np.float32)
    g = orc.make_grid((n, n, n), vs, mu, org)
    M, N = 300, 40
    pts = np.concatenate([rng.uniform(-0.2, 0.2, (M, 3)), np.ones((M, 1))], 1).astype(np.float32)
    pts[::17, 3] = 0
    pst = S.sample_pst(N, 99)
    pose = np.concatenate([Rotation.from_rotvec([0.2, -0.1, 0.3]).as_matrix(), [[0.37], [0.22], [0.52]]], 1).astype(np.float32)
    scale = np.array([0.1, 0.2, 0.15, 0.05, 0.1, 0.08], dtype=np.float32)
    got = orc.eval_particles(g, vol.reshape(-1), wgt.reshape(-1), pts, pst, pose, scale)
    M_O = int((pts[:, 3] != 0).sum())
    assert got["M_O"] == M_O
    Tc = pose.astype(np.float64)
    for j in range(N):
        dl = scale.astype(np.float64) * pst[j].astype(np.float64)
        qv = dl[:3]
        Rq = Rotation.from_quat([qv[0], qv[1], qv[2], math.sqrt(1 - qv @ qv)]).as_matrix()
        Rj, tj = Rq @ Tc[:, :3], Tc[:, 3] + dl[3:]
        Ssum, cnt = 0.0, 0
        for x in pts:
            if x[3] == 0:
                continue
            gg = ((Rj @ x[:3].astype(np.float64) + tj) - org) / np.float32(vs).astype(np.float64) - 0.5
            i0 = np.floor(gg).astype(int)
            if np.any(i0 < 0) or np.any(i0 + 1 > n - 1):
                continue
            f = gg - i0
            psi, good = 0.0, True
            for cz in (0, 1):
                for cy in (0, 1):
                    for cx in (0, 1):
                        if wgt[i0[2] + cz, i0[1] + cy, i0[0] + cx] <= 0:
                            good = False
                        wt = (f[0] if cx else 1 - f[0]) * (f[1] if cy else 1 - f[1]) * (f[2] if cz else 1 - f[2])
                        psi += wt * float(vol[i0[2] + cz, i0[1] + cy, i0[0] + cx])
            if good:
                Ssum += psi * psi
                cnt += 1
        assert got["n"][j] == cnt
        assert got["S"][j] == pytest.approx(Ssum, abs=1e-12)
        assert got["rho"][j] == pytest.approx(math.exp(-(Ssum + (M_O - cnt)) / M_O), abs=1e-12)


def test_p6_identity_optimal_on_noise_free_frame():
    """north_star: identity-pose fitness is optimal on noise-free synthetic frames (config-1 geometry)."""
    c = S.make_config1()
    g = orc.make_grid(c["dims"], c["voxel_size"], c["trunc"])
    clean = S.raycast_depth(c["scene"], c["pose"].astype(np.float64), c["K"], c["width"], c["height"]).astype(np.float32)
    pts = orc.backproject(clean, c["K"], 1).astype(np.float32)
    pst = np.concatenate([np.zeros((1, 6), np.float32), c["pst"]], 0)
    r = orc.eval_particles(g, c["tsdf"], c["weight"], pts, pst, c["pose"], c["scale"], nthreads=8)
    assert r["rho"][0] > 0.97
    assert np.all(r["rho"][0] > r["rho"][1:])
    assert int(np.argmax(r["rho"])) == 0


# ---------------------------------------------------------------------------------- O6  overlap mask
def test_o6_overlap_mask_geometry():
    w, h = 64, 48
    K = np.array([60.0, 60.0, 31.5, 23.5], dtype=np.float32)
    depth = np.full((h, w), 2.0, np.float32)
    depth[0, 0] = 0
    pts = orc.backproject(depth, K, 1)
    I = IDENT.astype(np.float64)
    keep, cnt = orc.overlap_mask(pts, I, I, K, w, h)
    assert cnt == w * h - 1 and keep[0] == 0 and keep[1] == 1         # same pose: every valid pixel re-projects onto itself
    # current camera translated by +0.5 m in x relative to the previous frame: a point at depth 2 m
    # moves by fx*0.5/2 = 15 px to the right in the previous image -> the 15 right-most columns drop
    T = I.copy()
    T[0, 3] = 0.5
    keep, cnt = orc.overlap_mask(pts, T, I, K, w, h)
    km = keep.reshape(h, w)
    assert np.all(km[1:, : w - 16] == 1) and np.all(km[:, w - 15 + 1:] == 0)
    # rotated by 180 degrees about y: everything is behind the previous camera
    T = np.array([[-1, 0, 0, 0], [0, 1, 0, 0], [0, 0, -1, 0]], dtype=np.float64)
    assert orc.overlap_mask(pts, T, I, K, w, h)[1] == 0


# ---------------------------------------------------------------------------------- P7  swarm update
def test_p7_hand_case():
    pst = np.array([[0.5, 0, 0, 0.2, 0, 0], [0, 0.4, 0, 0, -0.6, 0], [0.1, 0.1, 0.1, 0.1, 0.1, 0.1]], dtype=np.float32)
    rho = np.array([0.5, 0.7, 0.6, 0.4])
    r = np.array([0.1, 0.1, 0.1, 0.2, 0.2, 0.2])
    T = IDENT.astype(np.float64)
    o = orc.swarm_update(rho, pst, T, r)
    d1, d2 = r * pst[0].astype(np.float64), r * pst[1].astype(np.float64)
    dstar = (2 / 3) * d1 + (1 / 3) * d2
    assert o.n_aps == 2 and o.argmax == 1 and o.empty_run == 0
    assert np.allclose(list(o.delta_star), dstar, atol=1e-15)
    assert o.rho_tilde == pytest.approx((2 / 3) * 0.7 + (1 / 3) * 0.6, abs=1e-15)
    assert o.sum_omega == pytest.approx(0.3, abs=1e-15)
    rhat = (1 - o.rho_tilde) * np.abs(dstar) / np.linalg.norm(dstar) + 1e-3
    assert np.allclose(list(o.r_new), 0.1 * r + 0.9 * rhat, atol=1e-15)
    Tn = np.array(list(o.T_new)).reshape(3, 4)
    Rq = Rotation.from_quat([dstar[0], dstar[1], dstar[2], math.sqrt(1 - dstar[:3] @ dstar[:3])]).as_matrix()
    assert np.allclose(Tn[:, :3], Rq, atol=1e-14) and np.allclose(Tn[:, 3], dstar[3:], atol=1e-15)


def test_p7_empty_aps_and_stop_rules():
    pst = S.sample_pst(64, 3)
    T = np.concatenate([Rotation.random(random_state=5).as_matrix(), [[1.0], [2.0], [3.0]]], 1)
    r = np.full(6, 0.05)
    rho = np.full(65, 0.3)
    rho[0] = 0.6
    o = orc.swarm_update(rho, pst, T, r, empty_run=0)
    assert o.n_aps == 0 and o.empty_run == 1 and o.stop == 0 and o.argmax == 0
    assert np.allclose(np.array(list(o.T_new)).reshape(3, 4), T, atol=0)
    rhat = 2 * (1 - 0.6) / math.sqrt(6) + 1e-3           # P:L292 second corner case, isotropic
    assert np.allclose(list(o.r_new), 0.1 * 0.05 + 0.9 * rhat, atol=1e-15)
    o2 = orc.swarm_update(rho, pst, T, r, empty_run=1)
    assert o2.empty_run == 2 and o2.stop == 1
    # equal fitness is NOT an advantage (strict >), ties in argmax go to the lowest index
    rho[:] = 0.5
    o3 = orc.swarm_update(rho, pst, T, r)
    assert o3.n_aps == 0 and o3.argmax == 0
    # change below 1e-6 in all six dims -> stop code 2 (non-empty APS)
    tiny = np.full((4, 6), 1e-4, dtype=np.float32)
    o4 = orc.swarm_update(np.array([0.5, 0.6, 0.6, 0.6, 0.6]), tiny, T, np.full(6, 1e-3))
    assert o4.n_aps == 4 and o4.stop == 2


def test_p7_invariants_random():
    rng = np.random.default_rng(21)
    for trial in range(30):
        N = 200
        pst = S.sample_pst(N, 100 + trial)
        rho = rng.uniform(math.exp(-1), 1, N + 1)
        r = rng.uniform(1e-3, 0.3, 6)
        T = np.concatenate([Rotation.random(random_state=trial).as_matrix(), rng.normal(size=(3, 1))], 1)
        o = orc.swarm_update(rho, pst, T, r)
        aps = rho[1:] > rho[0]
        assert o.n_aps == aps.sum() and o.argmax == int(np.argmax(rho))
        if o.n_aps == 0:
            continue
        dl = r[None, :] * pst[aps].astype(np.float64)
        ds = np.array(list(o.delta_star))
        assert np.all(ds >= dl.min(0) - 1e-12) and np.all(ds <= dl.max(0) + 1e-12)      # convex hull (box) of APS
        assert rho[0] < o.rho_tilde <= rho[1:].max() + 1e-15
        rn = np.array(list(o.r_new))
        rhat = (rn - 0.1 * r) / 0.9
        assert np.all(rhat >= 1e-3 - 1e-12) and np.all(rhat <= 1 - math.exp(-1) + 1e-3 + 1e-12)
        assert np.linalg.norm((np.array(list(o.delta_star)) / r)) <= 1 + 1e-9       # A3: stays inside the PST ellipsoid


# ---------------------------------------------------------------------------------- ablation variants
def test_p7_rescale_variants_hand_case():
    """Fig. 11: Eq. (17) with its anisotropic part only, its isotropic part only, and both."""
    pst = np.array([[0.5, 0, 0, 0.2, 0, 0], [0, 0.4, 0, 0, -0.6, 0], [0.1, 0.1, 0.1, 0.1, 0.1, 0.1]], dtype=np.float32)
    rho = np.array([0.5, 0.7, 0.6, 0.4])
    r = np.array([0.1, 0.1, 0.1, 0.2, 0.2, 0.2])
    T = IDENT.astype(np.float64)
    dstar = (2 / 3) * r * pst[0].astype(np.float64) + (1 / 3) * r * pst[1].astype(np.float64)
    rt = (2 / 3) * 0.7 + (1 / 3) * 0.6
    full = orc.swarm_update(rho, pst, T, r)
    iso = orc.swarm_update(rho, pst, T, r, variant=orc.VAR_RESCALE_ISO)
    ani = orc.swarm_update(rho, pst, T, r, variant=orc.VAR_RESCALE_ANISO)
    for o in (iso, ani):        # only the axis lengths differ
        assert np.allclose(list(o.delta_star), list(full.delta_star), atol=0) and np.allclose(list(o.T_new), list(full.T_new), atol=0)
        assert o.rho_tilde == full.rho_tilde and o.n_aps == 2
    assert np.allclose(list(iso.r_new), 0.1 * r + 0.9 * ((1 - rt) / math.sqrt(6) + 1e-3), atol=1e-15)
    assert np.allclose(list(ani.r_new), 0.1 * r + 0.9 * (np.abs(dstar) / np.linalg.norm(dstar) + 1e-3), atol=1e-15)
    # the anisotropic direction is a unit vector; the full rule is the product of the two parts
    a = (np.array(list(ani.r_new)) - 0.1 * r) / 0.9 - 1e-3
    i = (np.array(list(iso.r_new)) - 0.1 * r) / 0.9 - 1e-3
    f = (np.array(list(full.r_new)) - 0.1 * r) / 0.9 - 1e-3
    assert np.linalg.norm(a) == pytest.approx(1.0, abs=1e-12)
    assert np.allclose(f, a * i * math.sqrt(6), atol=1e-15)
    # an empty advantage set has no direction: every variant falls back to the same rule
    rho0 = np.array([0.9, 0.7, 0.6, 0.4])
    base = list(orc.swarm_update(rho0, pst, T, r).r_new)
    for v in (orc.VAR_RESCALE_ISO, orc.VAR_RESCALE_ANISO, orc.VAR_NO_OVERLAP):
        assert list(orc.swarm_update(rho0, pst, T, r, variant=v).r_new) == base


def test_rho_no_normalize_closed_form():
    """ "No Normalize": Eq. (14) instead of Eq. (20).  rho_14 = rho_20 ^ |O|, and with psi = a/mu at every
    one of M points rho_14 = exp(-M (a/mu)^2)."""
    M, a_mu = 137, 0.25
    S_ = M * a_mu ** 2
    assert orc.rho(S_, M, M, 2) == pytest.approx(math.exp(-M * a_mu ** 2), rel=1e-14)
    assert orc.rho(S_, M, M, 2) == pytest.approx(orc.rho(S_, M, M, 0) ** M, rel=1e-12)
    assert orc.rho(3.0, 40, 50, 2) == pytest.approx(math.exp(-(3.0 + 10)), rel=1e-14)      # F2: unsampled points count 1
    assert orc.rho(1.0, 0, 0, 2) == 0.0


def test_no_overlap_variant_uses_every_valid_pixel():
    """ "No Overlap": O_k := I_d.  With the previous pose turned away, Eq. (19) keeps nothing while the
    variant keeps every valid pixel; with the previous pose = the current one the two coincide."""
    g = _grid()[0]
    F = np.full(32 ** 3, 0.5, np.float32); W = np.ones(32 ** 3, np.float32)
    K = np.array([40.0, 40.0, 15.5, 11.5], np.float32)
    depth = np.full((24, 32), 0.7, np.float32); depth[3, 4] = 0.0
    psts = [S.sample_pst(n, 40 + i) for i, n in enumerate((16, 16, 16))]
    T = np.array([[1, 0, 0, 0.0], [0, 1, 0, 0.0], [0, 0, 1, 0.1]], np.float32)
    away = np.array([[-1, 0, 0, 0.0], [0, 1, 0, 0.0], [0, 0, -1, 0.1]], np.float32)      # looks the other way
    kw = dict(r0=np.full(6, 0.01), early_stop=False)
    a = orc.pfo_track(g, F, W, depth, K, psts, (1, 2, 4), 3, T, away, **kw)
    b = orc.pfo_track(g, F, W, depth, K, psts, (1, 2, 4), 3, T, away, variant=orc.VAR_NO_OVERLAP, **kw)
    assert [t.M_O for t in a["trace"]] == [0, 0, 0]
    assert b["trace"][0].M_O == 24 * 32 - 1 and b["trace"][1].M_O == 12 * 16 and b["trace"][2].M_O == 6 * 8
    c = orc.pfo_track(g, F, W, depth, K, psts, (1, 2, 4), 1, T, T, **kw)
    d = orc.pfo_track(g, F, W, depth, K, psts, (1, 2, 4), 1, T, T, variant=orc.VAR_NO_OVERLAP, **kw)
    assert c["trace"][0].M_O == d["trace"][0].M_O == 24 * 32 - 1 and c["trace"][0].rho_ref == d["trace"][0].rho_ref


def test_p7_threshold_variant_hand_case_and_loop():
    """A14 variant: the advantage-set threshold is carried from the previous iteration instead of being
    re-evaluated.  Hand case on the update; then the loop: iteration 1 evaluates the centre exactly, iteration k > 1 uses
    Eq. (21)'s rho~ of iteration k-1, or after an empty step the threshold that step used."""
    pst = np.array([[0.5, 0, 0, 0.2, 0, 0], [0, 0.4, 0, 0, -0.6, 0], [0.1, 0.1, 0.1, 0.1, 0.1, 0.1]], dtype=np.float32)
    rho = np.array([0.5, 0.7, 0.6, 0.4])
    r = np.array([0.1, 0.1, 0.1, 0.2, 0.2, 0.2])
    T = IDENT.astype(np.float64)
    o = orc.swarm_update(rho, pst, T, r, variant=orc.VAR_THRESH_EQ21, thresh=0.65)      # only 0.7 beats 0.65
    assert o.n_aps == 1 and o.rho_ref == 0.65 and o.rho_tilde == pytest.approx(0.7, abs=1e-15)
    assert np.allclose(list(o.delta_star), r * pst[0].astype(np.float64), atol=1e-15) and o.argmax == 1
    e = orc.swarm_update(rho, pst, T, r, variant=orc.VAR_THRESH_EQ21, thresh=0.9)       # nothing beats 0.9
    assert e.n_aps == 0 and np.allclose(list(e.r_new), 0.1 * r + 0.9 * (2 * (1 - 0.9) / math.sqrt(6) + 1e-3), atol=1e-15)
    d = orc.swarm_update(rho, pst, T, r, variant=orc.VAR_THRESH_EQ21)                   # no carried value: rho[0]
    assert d.n_aps == 2 and d.rho_ref == 0.5
    assert orc.swarm_update(rho, pst, T, r, thresh=0.65).n_aps == 2                     # the flag, not the value, switches it on
    g, F, W, _, mu, vs = _plane_setup()
    K = np.array([60.0, 60.0, 31.5, 23.5], dtype=np.float32)
    depth = np.zeros((48, 64), dtype=np.float32)
    depth[6:42, 8:56] = 1.5
    T0 = IDENT.copy()
    T0[2, 3] = 0.05
    psts = [S.sample_pst(n, 60 + i) for i, n in enumerate((64, 96, 128))]
    kw = dict(r0=np.full(6, 0.04), early_stop=False)
    a = orc.pfo_track(g, F, W, depth, K, psts, (2, 4, 8), 6, T0, T0, **kw)
    b = orc.pfo_track(g, F, W, depth, K, psts, (2, 4, 8), 6, T0, T0, variant=orc.VAR_THRESH_EQ21, **kw)
    assert b["trace"][0].rho_ref == a["trace"][0].rho_ref            # first iteration: exact centre fitness in both
    for k in range(1, 6):
        prev = b["trace"][k - 1]
        assert b["trace"][k].rho_ref == (prev.rho_tilde if prev.n_aps > 0 else prev.rho_ref), k
    assert any(t.n_aps > 0 for t in b["trace"]) and any(x.rho_ref != y.rho_ref for x, y in zip(a["trace"][1:], b["trace"][1:]))


# ---------------------------------------------------------------------------------- baselines of Section 5.2
def test_baseline_propose_and_clamp_hand_case():
    """Eq. (12) as a random walk on the increments (B3, B4): float32 state, fp64 arithmetic, one rounding."""
    d = np.array([[0.1, -0.2, 0.05, 0.3, 0.0, -0.1], [0.0, 0.0, 0.0, 0.0, 0.0, 0.0], [0.6, 0.6, 0.5, 1.0, 2.0, 3.0]], dtype=np.float32)
    z = np.array([[1.0, -1.0, 0.5, 2.0, 0.0, 1.0], [0.0, 0.0, 0.0, 0.0, 0.0, 0.0], [0.0, 0.0, 0.0, 0.0, 0.0, 0.0]], dtype=np.float32)
    sg = np.array([0.01, 0.02, 0.03, 0.1, 0.2, 0.3], dtype=np.float32)
    out = orc.baseline_propose(d, None, sg, z)
    want0 = (d[0].astype(np.float64) + sg.astype(np.float64) * z[0].astype(np.float64)).astype(np.float32)
    assert np.array_equal(out[0], want0) and np.array_equal(out[1], d[1])
    q = out[2, :3].astype(np.float64)                   # |delta_q| = 0.98 > 0.95: radial clamp, translation untouched
    assert np.linalg.norm(q) == pytest.approx(0.95, abs=1e-7) and np.allclose(q / np.linalg.norm(q), d[2, :3] / np.linalg.norm(d[2, :3]), atol=1e-7)
    assert np.array_equal(out[2, 3:], d[2, 3:])
    anc = np.array([2, 2, 0], dtype=np.int32)           # ancestors: slots 0, 1 copy particle 2, slot 2 copies particle 0
    out2 = orc.baseline_propose(d, anc, np.zeros(6, np.float32), z)
    assert np.array_equal(out2[0], out[2]) and np.array_equal(out2[1], out[2]) and np.array_equal(out2[2], d[0])


def test_baseline_systematic_resampling_properties():
    """B1.  Closed-form properties of systematic resampling: every particle gets floor or ceil of N w copies; ancestors are
    non-decreasing; uniform weights give the identity; one non-zero weight takes every slot; unbiased over u."""
    rng = np.random.default_rng(17)
    N = 257
    w = rng.uniform(0.0, 1.0, N) ** 4
    wn = w / w.sum()
    for u in (0.0, 0.37, 0.999999):
        anc, _ = orc.systematic_resample(w, u)
        assert anc.shape == (N,) and np.all(np.diff(anc) >= 0) and anc.min() >= 0 and anc.max() < N
        cnt = np.bincount(anc, minlength=N)
        assert cnt.sum() == N and np.all(cnt >= np.floor(N * wn - 1e-9)) and np.all(cnt <= np.ceil(N * wn + 1e-9))
    assert np.array_equal(orc.systematic_resample(np.full(N, 0.3), 0.5)[0], np.arange(N))
    one = np.zeros(N); one[41] = 2.5
    assert np.all(orc.systematic_resample(one, 0.2)[0] == 41)
    mean = np.zeros(N)
    us = (np.arange(400) + 0.5) / 400
    for u in us:
        mean += np.bincount(orc.systematic_resample(w, u)[0], minlength=N)
    assert np.max(np.abs(mean / len(us) - N * wn)) < 0.01
    # `near` flags exactly the slots within tol of a boundary of the cumulative weights
    anc, near = orc.systematic_resample(w, 0.37, tol=1e-4)
    C = np.cumsum(wn)
    um = (np.arange(N) + 0.37) / N
    dist = np.min(np.abs(um[:, None] - np.concatenate([[0.0], C[:-1]])[None, :]), axis=1)
    assert np.array_equal(near.astype(bool), dist < 1e-4)


def test_baseline_pso_hand_case_and_best_bookkeeping():
    """B2: v <- omega v + c1 a (p - x) + c2 b (g - x), x <- x + v with the constriction constants of Clerc & Kennedy."""
    om, c = orc.pso_const(0), orc.pso_const(1)
    assert om == 0.7298 and c == 1.49618 and abs(om - 2 / abs(2 - 4.1 - math.sqrt(4.1 ** 2 - 4 * 4.1))) < 2e-4 and abs(c - om * 2.05) < 2e-4
    x = np.array([[0.1, 0.0, -0.1, 0.2, 0.3, 0.0]], dtype=np.float32)
    v = np.array([[0.01, 0.02, 0.0, -0.05, 0.0, 0.1]], dtype=np.float32)
    p = np.array([[0.2, 0.1, -0.1, 0.1, 0.3, 0.1]], dtype=np.float32)
    gb = np.array([0.0, 0.0, 0.0, 0.5, 0.5, 0.5, 0.9, 3.0], dtype=np.float32)
    a = np.array([[0.5, 0.25, 1.0, 0.0, 0.75, 0.5]], dtype=np.float32)
    b = np.array([[0.1, 0.2, 0.3, 0.4, 0.5, 0.6]], dtype=np.float32)
    x2, v2 = orc.baseline_pso_move(x, v, p, gb, a, b)
    X, V, P, G, A, B = (t.astype(np.float64) for t in (x[0], v[0], p[0], gb[:6], a[0], b[0]))
    vw = (om * V + c * A * (P - X) + c * B * (G - X)).astype(np.float32)
    assert np.allclose(v2[0], vw, rtol=0, atol=1e-9) and np.allclose(x2[0], (X + vw.astype(np.float64)).astype(np.float32), rtol=0, atol=1e-9)
    # bookkeeping: strict improvement, lowest index among equals
    fit = np.array([0.3, 0.8, 0.8, 0.1], dtype=np.float32)
    xs = np.arange(24, dtype=np.float32).reshape(4, 6)
    pb, pf, g8 = np.zeros((4, 6), np.float32), np.zeros(4, np.float32), np.zeros(8, np.float32)
    orc.baseline_best(fit, xs, pb, pf, True, g8)
    assert np.array_equal(pb, xs) and np.array_equal(pf, fit) and g8[6] == np.float32(0.8) and g8[7] == 1 and np.array_equal(g8[:6], xs[1])
    fit2 = np.array([0.5, 0.8, 0.7, 0.05], dtype=np.float32)
    orc.baseline_best(fit2, xs + 100, pb, pf, False, g8)
    assert np.array_equal(pf, np.array([0.5, 0.8, 0.8, 0.1], np.float32)) and np.array_equal(pb[0], xs[0] + 100) and np.array_equal(pb[1], xs[1])
    assert g8[7] == 1 and np.array_equal(g8[:6], xs[1])                    # 0.8 does not beat 0.8
    orc.baseline_best(np.array([0.1, 0.2, 0.95, 0.0], np.float32), xs - 50, None, None, False, g8)
    assert g8[7] == 2 and g8[6] == np.float32(0.95) and np.array_equal(g8[:6], xs[2] - 50)


def test_baseline_fitness_is_the_pinned_fitness_at_scale_one():
    """The baselines evaluate explicit increments: that is O5 with the template = the increments and unit axis lengths."""
    g, F, W, pts, mu, vs = _plane_setup()
    d = (0.05 * S.sample_pst(40, 5)).astype(np.float32)
    pose = np.concatenate([Rotation.from_rotvec([0.02, -0.01, 0.03]).as_matrix(), [[0.01], [0.0], [-0.02]]], 1).astype(np.float32)
    a = orc.eval_increments(g, F, W, pts, d, pose)
    b = orc.eval_particles(g, F, W, pts, d, pose, np.ones(6, np.float32))["rho"]
    assert np.array_equal(a, b) and a.min() < a.max()


# ---------------------------------------------------------------------------------- P8  whole loop (sanity)
def test_p8_pfo_recovers_a_perturbed_pose():
    """No paper value exists; sanity against synthetic ground truth on a reduced config-2 geometry:
    from a 10 deg / 6 cm offset the final error is far below the initial one within 20 iterations
    (consistent with "<10 iterations for fast motion")."""
    dims, vs, mu = (128, 128, 128), 0.02, 0.08
    scene = S.make_scene(4242, extent=2.56, inset=mu + 2 * vs, n_spheres=4, n_boxes=4, clearance=0.3)
    g = orc.make_grid(dims, vs, mu)
    w, h = 160, 120
    K = np.array([142.5, 142.5, 80.0, 60.0], dtype=np.float32)
    centre = 0.5 * (scene.room_lo + scene.room_hi)
    rng = np.random.Generator(np.random.Philox(77))
    pos = S.random_free_position(rng, scene, 0.35)
    T_prev = S.look_at(pos, centre + np.array([0.2, -0.1, -0.3]))
    F, W = orc.empty_volume(dims)
    for i in range(4):
        Ti = S.compose_delta(T_prev, [0, 0, 1], np.radians(-1.0 * (3 - i)), [0.01 * (i - 3), 0, 0])
        d = S.add_noise(S.raycast_depth(scene, Ti, K, w, h), 500 + i, sigma_rel=0.005)
        orc.integrate(g, F, W, d, K, Ti.astype(np.float32), nthreads=8)
    T_true = S.compose_delta(T_prev, [0.3, 0.5, 0.8], np.radians(10.0), [0.04, -0.03, 0.03])
    depth = S.add_noise(S.raycast_depth(scene, T_true, K, w, h), 600, sigma_rel=0.005)
    psts = [S.sample_pst(n, 700 + i) for i, n in enumerate((1024, 3072, 10240))]
    out = orc.pfo_track(g, F, W, depth, K, psts, (2, 4, 8), 20, T_prev, T_prev, r0=None, early_stop=False, nthreads=8)
    assert out["iters_run"] == 20 and len(out["trace"]) == 20
    e0 = np.linalg.norm(T_prev[:, 3] - T_true[:, 3])
    e1 = np.linalg.norm(out["pose"][:, 3] - T_true[:, 3])
    a0 = S.rotation_angle_deg(T_prev[:, :3], T_true[:, :3])
    a1 = S.rotation_angle_deg(out["pose"][:, :3], T_true[:, :3])
    assert e1 < 0.25 * e0 and a1 < 0.25 * a0, (e0, e1, a0, a1)
    tr = out["trace"]
    assert [t.level for t in tr[:6]] == [0, 1, 2, 0, 1, 2]                 # A15 resolution order
    assert tr[-1].rho_ref > tr[0].rho_ref                                 # fitness of the centre improved
    assert np.allclose(out["r1"], list(tr[0].r))                          # P:L286  r_0^{t+1} = r_1^t
    for t in tr:
        assert all(1e-3 * 0.9 <= x <= 1.0 for x in t.r)
    # early stop variant terminates no later and ends with a stop code
    out2 = orc.pfo_track(g, F, W, depth, K, psts, (2, 4, 8), 20, T_prev, T_prev, r0=None, early_stop=True, nthreads=8)
    assert out2["iters_run"] <= 20
    if out2["iters_run"] < 20:
        assert out2["trace"][-1].stop in (1, 2)


def test_p8_first_frame_rule_and_bookkeeping_closed_form():
    """A11 and the loop's counters, on the P6 plane where rho(T_0) is known in closed form.
    The camera starts a = 6 cm beyond the true pose along the plane normal, so every point has psi = -a/mu and
    rho(T_0) = exp(-(a/mu)^2); the first-frame rule must give r_0,d = 2 (1 - rho(T_0))/sqrt(6) + eps.  The three
    templates only move the camera further away (strictly worse), so every advantage set is empty: the pose must not
    move, r^ = 2 (1 - rho_ref)/sqrt(6) + eps = r_0 and hence r_1 = beta r_0 + (1 - beta) r^ = r_0 exactly -- any other
    r_0 would show up in r_1.  evals = |O| of the centre-only evaluation + sum_k (N_l + 1) |O_k|."""
    g, F, W, _, mu, vs = _plane_setup()
    w, h = 64, 48
    K = np.array([60.0, 60.0, 31.5, 23.5], dtype=np.float32)
    depth = np.zeros((h, w), dtype=np.float32)
    depth[6:42, 8:56] = 1.5                               # interior pixels only: their cells were all observed
    a = 0.06
    T0 = IDENT.copy()
    T0[2, 3] = a
    psts = [np.array([[0, 0, 0, 0, 0, s] for s in np.linspace(0.3, 1.0, n)], dtype=np.float32) for n in (3, 4, 5)]
    strides = (2, 4, 8)
    rho0 = math.exp(-(a / mu) ** 2)
    r0 = 2 * (1 - rho0) / math.sqrt(6) + 1e-3
    out = orc.pfo_track(g, F, W, depth, K, psts, strides, 3, T0, T0, r0=None, early_stop=False)
    M = [int((depth[s // 2::s, s // 2::s] > 0).sum()) for s in strides]
    tr = out["trace"]
    assert [t.M_O for t in tr] == M and [t.n_aps for t in tr] == [0, 0, 0] and [t.argmax for t in tr] == [0, 0, 0]
    assert [t.empty_run for t in tr] == [1, 2, 3] and [t.stop for t in tr] == [0, 1, 1]
    for t in tr:
        assert t.rho_ref == pytest.approx(rho0, rel=1e-6) and t.rho_max == t.rho_ref
        assert np.allclose(list(t.r), r0, rtol=1e-6)      # r_k = r_0 for every k
        assert np.array_equal(np.array(list(t.pose)).reshape(3, 4), T0.astype(np.float64))
    assert np.allclose(out["r1"], r0, rtol=1e-6)
    assert out["evals"] == M[0] + 4 * M[0] + 5 * M[1] + 6 * M[2]
    assert out["final_count"] == M[2] and out["final_rho"] == pytest.approx(rho0, rel=1e-6) and out["iters_run"] == 3
    # with the paper's stop rule the loop ends after the second empty advantage set
    es = orc.pfo_track(g, F, W, depth, K, psts, strides, 20, T0, T0, r0=None, early_stop=True)
    assert es["iters_run"] == 2 and es["trace"][-1].stop == 1 and es["evals"] == M[0] + 4 * M[0] + 5 * M[1]
    assert es["final_count"] == M[1]
    # a caller-supplied r_0 replaces the rule: r_1 = beta r_0 + (1 - beta) r^, and no centre-only evaluation is counted
    given = orc.pfo_track(g, F, W, depth, K, psts, strides, 1, T0, T0, r0=np.full(6, 0.02), early_stop=False)
    assert np.allclose(given["r1"], 0.1 * 0.02 + 0.9 * r0, rtol=1e-6) and given["evals"] == 4 * M[0]


def test_p8_oracle_tracks_the_config3_motion_against_ground_truth():
    """The readings taken for config 3 (12 cm truncation R-C3, search prior R-C3b, F2 normalisation A6, Eq. 19 overlap) against
    synthetic GROUND TRUTH, not against the CUDA path: five consecutive frames of the fast-motion sequence (10 cm and about
    5 degrees between frames, 1 % depth noise, 5 % dropout) on the 512^3 map fused from the twelve frames before them.
    Un-assisted (each frame starts from the previous estimate and r_1): every frame ends within 5 cm of the true position
    and at less than 0.4 of the distance it started from.  (Over the whole 200-frame sequence, whose rotations reach 20
    degrees per frame -- beyond the paper's fastest data, A25 -- the tracker does lose frames: bench.py --sequence reports
    that; this pin shows the readings do track the motion the paper evaluates.)"""
    scene = S.make_config3_scene()
    traj = S.make_config3_trajectory(scene, n_frames=200)
    dims, vs, mu = (512, 512, 512), 0.01, 0.12
    g = orc.make_grid(dims, vs, mu)
    F, W = orc.empty_volume(dims)
    K = None
    for i in range(18, 30):
        d, K = S.render_frame(scene, traj[i], 3, i)
        orc.integrate(g, F, W, d, K, traj[i].astype(np.float32), half_storage=True, nthreads=8)
    psts = [S.sample_pst(n, S.config_seed(3, 5 + i)) for i, n in enumerate((1024, 3072, 10240))]
    pose, r0 = traj[29].astype(np.float32), np.array([0.03, 0.03, 0.03, 0.15, 0.15, 0.15])
    for i in range(30, 35):
        d, _ = S.render_frame(scene, traj[i], 3, i)
        start = np.linalg.norm(pose[:, 3].astype(np.float64) - traj[i][:, 3])
        o = orc.pfo_track(g, F, W, d, K, psts, (8, 16, 32), 20, pose, pose, r0=r0, nthreads=8)
        te = np.linalg.norm(o["pose"][:, 3] - traj[i][:, 3])
        assert start > 0.09 and te < 0.05 and te < 0.4 * start, (i, start, te)
        assert S.rotation_angle_deg(o["pose"][:, :3], traj[i][:, :3]) < 2.0
        pose, r0 = o["pose"].astype(np.float32), o["r1"]
        orc.integrate(g, F, W, d, K, pose, half_storage=True, nthreads=8)


# ---- P9: ray-cast read-out (O9) against closed forms --------------------------------------------------------------
def _rc_world(n=48, vs=0.02):
    g = orc.make_grid((n, n, n), vs, 6 * vs, (0.0, 0.0, 0.0))
    c = _centres(n, vs, np.zeros(3))
    K = np.array([60.0, 60.0, 31.5, 23.5], dtype=np.float32)
    return g, c, K, 64, 48


def test_p9_raycast_plane_is_exact():
    """Trilinear interpolation reproduces an affine field, so the crossing of a plane is the ray/plane intersection to
    rounding wherever the two bracketing samples see unclipped corners; the normal is the plane's (towards the camera)."""
    n, vs = 48, 0.02
    g, c, K, w, h = _rc_world(n, vs)
    mu = 6 * vs
    nrm = np.array([0.2, -0.3, 1.0]); nrm /= np.linalg.norm(nrm)
    off = nrm @ np.array([0.48, 0.48, 0.6])
    tsdf = np.clip((off - c @ nrm) / mu, -1, 1).astype(np.float32)
    wgt = np.ones_like(tsdf)
    R = Rotation.from_euler("xyz", [4.0, -6.0, 10.0], degrees=True).as_matrix()
    pose = np.hstack([R, np.array([[0.45], [0.5], [0.1]])]).astype(np.float32)
    depth, normals, frag = orc.raycast(g, tsdf, wgt, K, w, h, pose, 0.03, 2.0)
    P = pose.astype(np.float64)
    v, u = np.mgrid[0:h, 0:w]
    dc = np.stack([(u - K[2]) / K[0], (v - K[3]) / K[1], np.ones_like(u, dtype=np.float64)], -1)
    dw = dc @ P[:, :3].T
    z_exact = (off - nrm @ P[:, 3]) / (dw @ nrm)
    hit = P[:, 3] + dw * z_exact[..., None]
    inside = np.all((hit > 4 * vs) & (hit < (n - 4) * vs), axis=-1)
    assert inside.sum() > 0.3 * w * h
    assert np.max(np.abs(depth[inside] - z_exact[inside])) < 1e-6        # fp32 TSDF samples of an affine field
    assert np.max(np.abs(normals[inside] + nrm)) < 1e-5
    # a camera that looks away from the grid sees nothing
    back = pose.copy()
    back[:, :3] = pose[:, :3] @ np.diag([-1.0, 1.0, -1.0]).astype(np.float32)
    d0, n0, _ = orc.raycast(g, tsdf, wgt, K, w, h, back, 0.03, 2.0)
    assert np.all(d0 == 0) and np.all(np.isnan(n0))
    # a march that ends before the plane finds nothing
    d2, _, _ = orc.raycast(g, tsdf, wgt, K, w, h, pose, 0.03, 0.3, want_normals=False)
    assert np.all(d2 == 0)


def test_p9_raycast_sphere_backface_and_unobserved():
    n, vs = 48, 0.02
    g, c, K, w, h = _rc_world(n, vs)
    mu = 6 * vs
    ctr, rad = np.array([0.48, 0.48, 0.55]), 0.25
    tsdf = np.clip((np.linalg.norm(c - ctr, axis=1) - rad) / mu, -1, 1).astype(np.float32)
    wgt = np.ones_like(tsdf)
    pose = np.hstack([np.eye(3), np.array([[0.48], [0.48], [-0.2]])]).astype(np.float32)
    depth, normals, _ = orc.raycast(g, tsdf, wgt, K, w, h, pose, 0.03, 2.0)
    v, u = np.mgrid[0:h, 0:w]
    dc = np.stack([(u - K[2]) / K[0], (v - K[3]) / K[1], np.ones_like(u, dtype=np.float64)], -1)
    o = pose[:, 3].astype(np.float64) - ctr
    a, b, cc = (dc * dc).sum(-1), 2 * (dc @ o), o @ o - rad * rad
    disc = b * b - 4 * a * cc
    z_exact = np.where(disc > 0, (-b - np.sqrt(np.maximum(disc, 0))) / (2 * a), 0)
    core = disc > 0.04 * (b * b)                # away from the silhouette
    assert core.sum() > 200
    assert np.max(np.abs(depth[core] - z_exact[core])) < 0.15 * vs       # O(vs^2 / radius) interpolation error
    hitp = pose[:, 3].astype(np.float64) + dc * depth[..., None]
    want_n = (hitp - ctr) / np.linalg.norm(hitp - ctr, axis=-1, keepdims=True)
    cosang = np.sum(normals[core] * want_n[core], axis=-1)
    assert np.min(cosang) > math.cos(math.radians(1.0))
    assert np.all(depth[disc < -0.01 * b * b] == 0)                     # rays that miss the ball
    # from inside the ball the first sign change is negative -> positive: not a surface
    pose_in = np.hstack([np.eye(3), ctr.reshape(3, 1)]).astype(np.float32)
    d_in, _, _ = orc.raycast(g, tsdf, wgt, K, w, h, pose_in, 0.03, 2.0, want_normals=False)
    assert np.all(d_in == 0)
    # an unobserved slab over the near surface: the crossing has an invalid neighbour sample -> no hit there
    w3 = wgt.reshape(n, n, n).copy()            # [z, y, x]
    w3[12:20, :, :] = 0                         # z in [0.24, 0.40): the front cap (surface at z = 0.30)
    d_gap, _, _ = orc.raycast(g, tsdf, w3.reshape(-1), K, w, h, pose, 0.03, 2.0, want_normals=False)
    centre = (np.abs(u - K[2]) < 4) & (np.abs(v - K[3]) < 4)
    assert np.all(depth[centre] > 0) and np.all(d_gap[centre] == 0)


# ---- P10: surface point set (O10) against closed forms ------------------------------------------------------------
def test_p10_surface_points_plane_exact_sphere_count_and_unobserved():
    """Plane: trilinear / linear interpolation is exact on an affine field, so every point lies ON the plane and there is
    exactly one per crossing edge (counted independently).  Sphere: points within the linear-interpolation error
    vs^2 / (8 R) (+ rounding) of the sphere, and their number is the lattice-edge crossing count of a closed surface,
    (1 / vs^2) * integral of (|n_x| + |n_y| + |n_z|) dA = 6 pi R^2 / vs^2, to 2 %.  Unobserved samples carry no point."""
    n, vs = 48, 0.02
    g = orc.make_grid((n, n, n), vs, 6 * vs, (0.1, -0.2, 0.05))
    c = _centres(n, vs, np.array([0.1, -0.2, 0.05]))
    mu = 6 * vs
    nrm = np.array([0.3, -0.2, 1.0]); nrm /= np.linalg.norm(nrm)
    off = nrm @ (np.array([0.1, -0.2, 0.05]) + np.array([0.48, 0.47, 0.52]))
    field = ((off - c @ nrm) / mu).astype(np.float32)            # affine, NOT clamped: the interpolation is then exact
    wgt = np.ones_like(field)
    pts, edge = orc.surface_points(g, field, wgt)
    assert np.max(np.abs(pts @ nrm - off)) < 2e-7                # float32 field values: 1e-7 relative
    F3 = field.reshape(n, n, n)                                  # [z, y, x]
    pos = F3 > 0
    want = int((pos[:, :, :-1] != pos[:, :, 1:]).sum() + (pos[:, :-1, :] != pos[:, 1:, :]).sum() + (pos[:-1, :, :] != pos[1:, :, :]).sum())
    assert len(pts) == want > 3000 and len(np.unique(edge)) == want and np.all(np.diff(edge) > 0)
    axis = edge % 3
    a_lin = edge // 3
    ca = c[a_lin]
    rest = np.ones((len(pts), 3), bool); rest[np.arange(len(pts)), axis] = False
    assert np.allclose(pts[rest], ca[rest], atol=1e-12)          # the point moves along its edge only ...
    tt = (pts - ca)[np.arange(len(pts)), axis] / np.float32(vs)
    assert np.all(tt >= -1e-9) and np.all(tt <= 1 + 1e-9)         # ... and stays on it
    # sphere
    R, ctr = 0.3, np.array([0.1, -0.2, 0.05]) + 0.48
    sph = np.clip((np.linalg.norm(c - ctr, axis=1) - R) / mu, -1, 1).astype(np.float32)      # positive outside (free space)
    pts, edge = orc.surface_points(g, sph, wgt)
    err = np.abs(np.linalg.norm(pts - ctr, axis=1) - R)
    assert err.max() < vs ** 2 / (8 * R) * 1.5 + 1e-6
    assert abs(len(pts) - 6 * math.pi * R ** 2 / vs ** 2) < 0.02 * 6 * math.pi * R ** 2 / vs ** 2
    # unobserved: blank a slab through the sphere; no point may touch a blanked voxel
    w2 = wgt.copy().reshape(n, n, n); w2[:, 20:26, :] = 0
    pts2, edge2 = orc.surface_points(g, sph, w2.reshape(-1))
    a2 = edge2 // 3
    b2 = a2 + np.array([1, n, n * n])[edge2 % 3]
    assert 0 < len(pts2) < len(pts) and np.all(w2.reshape(-1)[a2] > 0) and np.all(w2.reshape(-1)[b2] > 0)
    # a value of exactly zero counts as "not positive": the crossing sits on the sample
    z = np.ones(n ** 3, np.float32); z[n * n * 10 + n * 10 + 10] = 0.0
    p0, e0 = orc.surface_points(g, z, wgt)
    assert len(p0) == 6 and np.allclose(p0, c[n * n * 10 + n * 10 + 10], atol=1e-12)


# ---- P11: Gauss-Newton SDF tracker (O11) -----------------------------------------------------------------------------
def test_p11_gauss_newton_closed_forms():
    """(1) The derivative of the trilinear interpolant of an affine field is that field's gradient.  (2) Three orthogonal
    planes (a room corner) fix all six degrees of freedom and the TSDF is affine near each wall, so Gauss-Newton converges
    quadratically: from 3 cm / 2 degrees off the cost falls 120 -> 8e-3 -> 1e-11 and the pose is recovered to 1e-7.
    (3) One wall only: the cost before the step is M (a / mu)^2 for a normal offset a, and the rank-3 normal equations are
    either reported singular (pose unchanged) or solved by a step that removes the offset."""
    n, vs = 12, 0.125
    org = np.array([0.25, -0.5, 1.0])
    g = orc.make_grid((n, n, n), vs, 0.375, org)
    a3 = np.array([0.31, -0.17, 0.23])
    ii, jj, kk = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    cen = org + (np.stack([ii, jj, kk], -1) + 0.5) * vs
    field = np.zeros(n ** 3, dtype=np.float32)
    field[(ii + n * (jj + n * kk)).reshape(-1)] = (cen.reshape(-1, 3) @ a3 + 0.05)
    ok, psi, gr = orc.trilinear_grad(g, field, np.ones(n ** 3, np.float32), org + np.array([0.7, 0.66, 0.81]))
    assert ok and np.allclose(gr, a3, atol=1e-6) and psi == pytest.approx((org + np.array([0.7, 0.66, 0.81])) @ a3 + 0.05, abs=1e-6)
    # room corner: psi = min over three walls of the distance to the wall / mu, sampled on the grid (exactly affine near each wall)
    n, vs, mu = 64, 0.02, 0.1
    g = orc.make_grid((n, n, n), vs, mu, (0.0, 0.0, 0.0))
    c = _centres(n, vs, np.zeros(3))
    walls = np.array([0.2, 0.25, 0.3])                              # planes x = 0.2, y = 0.25, z = 0.3; free space beyond them
    tsdf = np.clip(np.min(c - walls, axis=1) / mu, -1, 1).astype(np.float32)
    wgt = np.ones_like(tsdf)
    rng = np.random.default_rng(3)
    pts = []
    for ax in range(3):                                             # world points ON each wall, away from the edges
        p = rng.uniform(0.5, 1.0, (400, 3)); p[:, ax] = walls[ax]
        pts.append(p)
    P = np.concatenate(pts)
    T_true = np.concatenate([Rotation.from_rotvec([0.3, -0.2, 0.5]).as_matrix(), [[0.6], [0.7], [0.65]]], 1)
    X = (P - T_true[:, 3]) @ T_true[:, :3]                          # the same points in the camera frame
    points = np.concatenate([X, np.ones((len(X), 1))], 1).astype(np.float32)
    dR = Rotation.from_rotvec(np.radians(2.0) * np.array([0.6, -0.64, 0.48])).as_matrix()
    T0 = np.concatenate([dR @ T_true[:, :3], (dR @ T_true[:, 3] + np.array([0.02, -0.015, 0.018]))[:, None]], 1)
    out = orc.gn_track(g, tsdf, wgt, points, T0, 8)
    costs = [r.cost for r in out["rows"]]
    assert out["iters_run"] <= 4 and costs[0] > 50.0 and costs[1] < 1e-3 * costs[0] and costs[2] < 1e-6 * costs[1]
    assert np.max(np.abs(out["pose"] - T_true)) < 1e-7 and out["rows"][0].n == len(points)
    assert out["rows"][0].step_norm == pytest.approx(np.linalg.norm(np.linalg.solve(
        np.array(out["rows"][0].A).reshape(6, 6), -np.array(out["rows"][0].b))), rel=1e-9)
    # one wall only: a pure offset along its normal is removed by ONE step (the objective is quadratic there)
    px = rng.uniform(0.5, 1.0, (300, 3)); px[:, 0] = walls[0]
    pts1 = np.concatenate([px, np.ones((300, 1))], 1).astype(np.float32)
    I = np.concatenate([np.eye(3), np.zeros((3, 1))], 1)
    Ta = I.copy(); Ta[0, 3] = 0.03
    one = orc.gn_track(g, tsdf, wgt, pts1, Ta, 1)
    assert one["rows"][0].cost == pytest.approx(300 * (0.03 / mu) ** 2, rel=1e-5)
    # the normal equations of a single plane have rank 3 (normal translation + two tilts); the pivoted solve either reports
    # the singular system (pose unchanged) or, through rounding, a finite step that still removes the normal offset
    assert one["iters_run"] == 1 and (np.array_equal(one["pose"], Ta) or abs(one["pose"][0, 3]) < 1e-6)

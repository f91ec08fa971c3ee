"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star; DESIGN.md section 7 "Parity gates and tolerances"):
  fitness  relative 1e-5 (fp32 volume) / 2e-3 (fp16 volume), widened by fragile_j / M_O (A26)
  counts   exact up to the oracle's fragile count of that candidate (A26), expected 0 almost everywhere
  argmax   identical wherever the margin over the runner-up exceeds the tolerance (A18)
  TSDF     1e-4 * voxel_size (= 1e-4 * vs / trunc normalised) for fp32 storage; for fp16 storage <= 1 fp16
           ulp on <= 0.1 % of voxels and bit-equal elsewhere (A17); weights exact.
"""
import math

import numpy as np
import pytest

import oracle as orc
import rf_synth as S
from gates import check_integration

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

FIT_TOL = {0: 1e-5, 1: 2e-3}      # by rf dtype


def _rf():
    import paper_2105_05600_b200 as rf
    return rf


def _dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


IDENT = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0]], dtype=np.float32)


def _check_fitness(got_fit, got_cnt, ref, tol):
    fit = got_fit.cpu().numpy().astype(np.float64)
    cnt = got_cnt.cpu().numpy()
    M_O = max(ref["M_O"], 1)
    dn = np.abs(cnt.astype(np.int64) - ref["n"])
    assert np.all(dn <= ref["fragile"]), (dn.max(), ref["fragile"].max())
    rel = np.abs(fit - ref["rho"]) / np.maximum(ref["rho"], 1e-30)
    allowed = tol + 2.0 * ref["fragile"] / M_O
    assert np.all(rel <= allowed), (rel.max(), np.argmax(rel))
    # best particle identical wherever its margin over the runner-up exceeds the tolerance
    order = np.argsort(-ref["rho"], kind="stable")
    if len(order) > 1 and ref["rho"][order[0]] - ref["rho"][order[1]] > 2 * tol * ref["rho"][order[0]]:
        assert int(np.argmax(fit)) == int(order[0])
    return rel.max(), int((ref["fragile"] > 0).sum())


# ---------------------------------------------------------------------------------- a7 upload / download
@pytest.mark.parametrize("dtype", [0, 1])
def test_upload_download_roundtrip_ragged_dims(dtype):
    rf = _rf()
    dims = (21, 9, 13)                                  # not multiples of the 8^3 brick
    rng = np.random.default_rng(1)
    n = dims[0] * dims[1] * dims[2]
    t = rng.uniform(-1, 1, n).astype(np.float32)
    if dtype == 1:
        t = t.astype(np.float16).astype(np.float32)
    w = rng.integers(0, 4, n).astype(np.float32)
    vol = rf.Volume(dims, 0.02, 0.06, dtype=dtype)
    t0, w0 = vol.download()
    assert np.all(t0 == 1.0) and np.all(w0 == 0)        # fresh volume: unobserved everywhere
    vol.upload(t, w)
    t1, w1 = vol.download()
    assert np.array_equal(w1, w)
    assert np.array_equal(t1[w > 0], t[w > 0]) and np.all(t1[w == 0] == 1.0)
    vol.reset()
    t2, w2 = vol.download()
    assert np.all(t2 == 1.0) and np.all(w2 == 0)
    vol.destroy()


# ---------------------------------------------------------------------------------- a0 back-projection
@pytest.mark.parametrize("stride", [1, 4, 8, 32])
def test_backproject_matches_oracle(stride):
    rf = _rf()
    c = S.make_config1()
    depth = c["depth"].copy()
    depth[3, 5] = 0.0
    depth[7, 9] = np.nan
    vol = rf.Volume((8, 8, 8), 0.02, 0.06)
    pts = vol.backproject(_dev(depth), c["K"], stride).cpu().numpy()
    ref = orc.backproject(depth, c["K"], stride)
    assert pts.shape == ref.shape
    assert np.array_equal(pts[:, 3], ref[:, 3])
    assert np.allclose(pts[:, :3], ref[:, :3], rtol=3e-7, atol=1e-9)
    vol.destroy()


# ---------------------------------------------------------------------------------- config 1 (a2 + a3)
def test_config1_fitness_parity():
    rf = _rf()
    c = S.make_config1()
    g = orc.make_grid(c["dims"], c["voxel_size"], c["trunc"])
    vol = rf.Volume(c["dims"], c["voxel_size"], c["trunc"], dtype=rf.RF_F32_W8)
    vol.upload(c["tsdf"], c["weight"])
    pts = vol.backproject(_dev(c["depth"]), c["K"], 1)
    assert pts.shape[0] == 4800
    pst = np.concatenate([np.zeros((1, 6), np.float32), c["pst"]], 0)        # zero particle appended (centre)
    fit, cnt, Sraw = vol.eval_particles(pts, _dev(pst), c["pose"], c["scale"], return_S=True)
    ref = orc.eval_particles(g, c["tsdf"], c["weight"], pts.cpu().numpy(), pst, c["pose"], c["scale"], nthreads=8)
    worst, nfrag = _check_fitness(fit, cnt, ref, FIT_TOL[0])
    assert nfrag <= 8
    assert np.allclose(Sraw.cpu().numpy(), ref["S"], rtol=2e-5, atol=1e-4)
    # F1 normalisation shares S and n
    fit1, cnt1 = vol.eval_particles(pts, _dev(pst), c["pose"], c["scale"], mode=1)
    ref1 = orc.eval_particles(g, c["tsdf"], c["weight"], pts.cpu().numpy(), pst, c["pose"], c["scale"], mode=1, nthreads=8)
    _check_fitness(fit1, cnt1, ref1, FIT_TOL[0])
    # the paper's Poisson-disk template through the same gate, and Eq. (14) (mode 2)
    pp = np.concatenate([np.zeros((1, 6), np.float32), S.sample_pst_poisson(1024, S.config_seed(1, 6))], 0)
    fitp, cntp = vol.eval_particles(pts, _dev(pp), c["pose"], c["scale"])
    refp = orc.eval_particles(g, c["tsdf"], c["weight"], pts.cpu().numpy(), pp, c["pose"], c["scale"], nthreads=8)
    _check_fitness(fitp, cntp, refp, FIT_TOL[0])
    fit2, cnt2 = vol.eval_particles(pts, _dev(pst), c["pose"], c["scale"], mode=2)
    ref2 = orc.eval_particles(g, c["tsdf"], c["weight"], pts.cpu().numpy(), pst, c["pose"], c["scale"], mode=2, nthreads=8)
    assert np.array_equal(cnt2.cpu().numpy(), cnt.cpu().numpy())
    big = ref2["rho"] > 1e-30                                               # float32 output underflows below that
    assert np.allclose(fit2.cpu().numpy()[big], ref2["rho"][big], rtol=FIT_TOL[0] * ref2["M_O"])
    vol.destroy()


# ---------------------------------------------------------------------------------- ragged, partially observed
def _small_world(dims=(70, 66, 50), vs=0.03, mu=0.09, n_frames=3, seed=5150, half=False):
    scene = S.make_scene(seed, extent=dims[0] * vs, inset=mu + 2 * vs, n_spheres=2, n_boxes=2, clearance=0.3)
    scene.room_hi = np.array([dims[0] * vs, dims[1] * vs, dims[2] * vs]) - (mu + 2 * vs)
    w, h = 96, 72
    K = np.array([80.0, 80.0, 47.5, 35.5], dtype=np.float32)
    rng = np.random.Generator(np.random.Philox(seed))
    centre = 0.5 * (scene.room_lo + scene.room_hi)
    pos = centre + np.array([0.3, -0.2, 0.1])
    poses, frames = [], []
    for i in range(n_frames):
        T = S.look_at(pos + 0.02 * i * np.array([1, 0.5, 0]), centre + np.array([-0.6, 0.5, -0.2]) + 0.05 * i)
        d = S.add_noise(S.raycast_depth(scene, T, K, w, h), seed + i, sigma_rel=0.01, dropout=0.05)
        poses.append(T.astype(np.float32))
        frames.append(d)
    return scene, K, w, h, poses, frames


@pytest.mark.parametrize("dtype", [0, 1])
def test_integrate_parity_ragged(dtype):
    """Ragged volume, noisy frames with dropout; teacher-forced per frame (A21): both sides fuse frame i into the oracle's
    state after frame i-1.  Gate: tests/gates.py (weights exact off the oracle's fragile voxels, R-I2)."""
    rf = _rf()
    dims, vs, mu = (70, 66, 50), 0.03, 0.09
    scene, K, w, h, poses, frames = _small_world(dims, vs, mu)
    g = orc.make_grid(dims, vs, mu)
    F, W = orc.empty_volume(dims)
    vol = rf.Volume(dims, vs, mu, dtype=dtype)
    for i, (T, d) in enumerate(zip(poses, frames)):
        Fprev, Wprev = F.copy(), W.copy()
        frag = np.zeros(F.size, dtype=np.uint8)
        orc.integrate(g, F, W, d, K, T, half_storage=(dtype == 1), nthreads=8, fragile=frag)
        vol.upload(Fprev, Wprev)
        vol.integrate(_dev(d), K, T)
        Ft, Wt = vol.download()
        ff, _, _ = check_integration(Ft, Wt, F, W, Wprev, frag, dtype == 1, vs, mu, tag=i)
        assert ff < 0.02
        assert abs(vol.last_updated() - int((W != Wprev).sum())) <= int(frag.sum())
    assert (W > 0).mean() > 0.03          # non-vacuity guard only: ~5 % of this volume (11 k voxels) is observed
    vol.destroy()


@pytest.mark.parametrize("dtype", [0, 1])
def test_integrate_parity_frustum_boundary(dtype):
    """Constant-depth frames from seeded poses inside and outside the grid: every voxel in front of the depth plane and
    inside the image updates, so the set of updated voxels IS the frustum and its boundary cuts through many bricks.
    Exercises both code paths of k_update (bricks strictly inside the frustum skip the per-voxel in-image tests, the
    others do not): weights must match the oracle exactly on the whole volume, off the oracle's fragile voxels."""
    rf = _rf()
    dims, vs, mu = (64, 56, 72), 0.04, 0.12
    w, h = 160, 120
    K = np.array([120.0, 118.0, 79.5, 59.5], dtype=np.float32)
    g = orc.make_grid(dims, vs, mu)
    F, W = orc.empty_volume(dims)
    vol = rf.Volume(dims, vs, mu, dtype=dtype)
    rng = np.random.Generator(np.random.Philox(77123))
    ext = np.array(dims) * vs
    for i in range(6):
        pos = rng.uniform(-0.3, 1.3, 3) * ext                     # some cameras sit outside the grid
        target = rng.uniform(0.2, 0.8, 3) * ext
        T = S.look_at(pos, target).astype(np.float32)
        d = np.full((h, w), 1.0 + 0.5 * i, dtype=np.float32)
        d[rng.random((h, w)) < 0.03] = 0.0                        # dropout: holes inside the frustum
        Fprev, Wprev = F.copy(), W.copy()
        frag = np.zeros(F.size, dtype=np.uint8)
        orc.integrate(g, F, W, d, K, T, half_storage=(dtype == 1), nthreads=8, fragile=frag)
        vol.upload(Fprev, Wprev)
        vol.integrate(_dev(d), K, T)
        Ft, Wt = vol.download()
        ff, _, _ = check_integration(Ft, Wt, F, W, Wprev, frag, dtype == 1, vs, mu, tag=i)
        assert ff < 0.02
    assert (W > 0).mean() > 0.3           # the frusta cover a large part of the grid
    vol.destroy()


def test_integrate_parity_image_size_that_disables_the_biased_pixel_path():
    """k_update's inside-frustum path indexes the frame through biased pixel coordinates, which needs
    0x4B400000 * (w + 1) mod 2^32 + w * h <= 2^32; 2394 x 1754 is a size where that fails, so the library must fall back
    to the general path for every brick.  Weights exact and values within tolerance against the oracle."""
    rf = _rf()
    w, h = 2394, 1754
    assert (0x4B400000 * (w + 1)) % (1 << 32) + w * h > (1 << 32)
    dims, vs, mu = (48, 40, 56), 0.05, 0.15
    K = np.array([1500.0, 1500.0, 1196.5, 876.5], dtype=np.float32)
    g = orc.make_grid(dims, vs, mu)
    F, W = orc.empty_volume(dims)
    vol = rf.Volume(dims, vs, mu, dtype=0)
    ext = np.array(dims) * vs
    T = S.look_at(np.array([0.1, 0.2, -0.3]) * ext, np.array([0.6, 0.5, 0.7]) * ext).astype(np.float32)
    d = np.full((h, w), 2.5, dtype=np.float32)
    d[::7, ::5] = 0.0
    Wprev = W.copy()
    frag = np.zeros(F.size, dtype=np.uint8)
    orc.integrate(g, F, W, d, K, T, half_storage=False, nthreads=8, fragile=frag)
    vol.integrate(_dev(d), K, T)
    Ft, Wt = vol.download()
    ff, _, _ = check_integration(Ft, Wt, F, W, Wprev, frag, False, vs, mu)
    assert (W > 0).mean() > 0.2 and ff < 0.05          # 1500-pixel focal length: a pixel is 1.7 mm wide at 2.5 m
    vol.destroy()


def test_integrate_parity_wide_angle_depth_step_at_the_image_border():
    """Far cull, wide field of view (fx = w/2: 90 degrees): an off-axis brick's silhouette is wider than its on-axis one,
    and at a depth discontinuity near the image border a brick must be tested against every tile it can project onto.
    Near wall in the centre, far wall in a band along the border: bricks behind the near wall that also see the far band
    have to be swept."""
    rf = _rf()
    dims, vs, mu = (96, 96, 96), 0.05, 0.15
    w, h = 160, 120
    K = np.array([80.0, 80.0, 79.5, 59.5], dtype=np.float32)
    g = orc.make_grid(dims, vs, mu)
    vol = rf.Volume(dims, vs, mu, dtype=0)
    ext = np.array(dims) * vs
    rng = np.random.Generator(np.random.Philox(424242))
    for i, band in enumerate((6, 17, 30)):
        F, W = orc.empty_volume(dims)
        d = np.full((h, w), 0.9 + 0.2 * i, dtype=np.float32)      # near surface
        d[:, :band] = 4.3; d[:, w - band:] = 4.0; d[:band, :] = 3.7; d[h - band:, :] = 4.4      # far surface along the border
        pos = np.array([0.5, 0.5, 0.08]) * ext + rng.uniform(-0.1, 0.1, 3)
        T = S.look_at(pos, np.array([0.5, 0.55, 0.9]) * ext + rng.uniform(-0.3, 0.3, 3)).astype(np.float32)
        Wprev = W.copy()
        frag = np.zeros(F.size, dtype=np.uint8)
        orc.integrate(g, F, W, d, K, T, nthreads=8, fragile=frag)
        vol.reset()
        vol.integrate(_dev(d), K, T)
        Ft, Wt = vol.download()
        check_integration(Ft, Wt, F, W, Wprev, frag, False, vs, mu, tag=band)
        assert (W > 0).mean() > 0.03
    vol.destroy()


def test_integrate_host_depth_equals_device_depth():
    rf = _rf()
    dims, vs, mu = (40, 40, 40), 0.05, 0.15
    scene, K, w, h, poses, frames = _small_world((70, 66, 50), 0.03, 0.09, n_frames=1)
    a, b = rf.Volume(dims, vs, mu), rf.Volume(dims, vs, mu)
    a.integrate(_dev(frames[0]), K, poses[0])
    b.integrate(frames[0], K, poses[0])                  # host buffer: H2D copy inside the call
    ta, wa = a.download()
    tb, wb = b.download()
    assert np.array_equal(ta, tb) and np.array_equal(wa, wb) and (wa > 0).sum() > 100
    # depth_on_host == 2: fuse the frame the previous host-depth call staged on the device
    b.integrate(None, K, poses[0], staged_shape=frames[0].shape)
    a.integrate(_dev(frames[0]), K, poses[0])
    assert all(np.array_equal(x, y) for x, y in zip(a.download(), b.download()))
    with pytest.raises(rf.RFError):
        a.integrate(None, K, poses[0], staged_shape=frames[0].shape)      # nothing staged on this volume
    with pytest.raises(rf.RFError):
        b.integrate(None, K, poses[0], staged_shape=(h + 1, w))           # staged frame has another size
    a.destroy(); b.destroy()


@pytest.mark.parametrize("dtype,M,N", [(0, 1000, 777), (1, 1000, 777), (1, 31, 5), (0, 4097, 129)])
def test_fitness_parity_partially_observed_ragged(dtype, M, N):
    rf = _rf()
    dims, vs, mu = (70, 66, 50), 0.03, 0.09
    scene, K, w, h, poses, frames = _small_world(dims, vs, mu)
    g = orc.make_grid(dims, vs, mu)
    F, W = orc.empty_volume(dims)
    for T, d in zip(poses, frames):
        orc.integrate(g, F, W, d, K, T, half_storage=(dtype == 1), nthreads=8)
    vol = rf.Volume(dims, vs, mu, dtype=dtype)
    vol.upload(F, W)
    T_eval = S.compose_delta(poses[-1].astype(np.float64), [0.2, 0.9, 0.1], np.radians(3.0), [0.02, -0.01, 0.015])
    d = S.add_noise(S.raycast_depth(scene, T_eval, K, w, h), 777, sigma_rel=0.01, dropout=0.05)
    pts_all = orc.backproject(d, K, 1).astype(np.float32)
    rng = np.random.Generator(np.random.Philox(99))
    sel = np.sort(rng.choice(pts_all.shape[0], M, replace=False))
    pts = np.ascontiguousarray(pts_all[sel])
    pst = S.sample_pst(N, 4321)
    scale = np.array([0.03, 0.05, 0.02, 0.04, 0.06, 0.03], dtype=np.float32)
    pose = poses[-1]
    fit, cnt = vol.eval_particles(_dev(pts), _dev(pst), pose, scale)
    ref = orc.eval_particles(g, F, W, pts, pst, pose, scale, nthreads=8)
    assert 0 < ref["n"].max() and ref["n"].min() < ref["M_O"]          # unobserved / out-of-grid cells are exercised
    _check_fitness(fit, cnt, ref, FIT_TOL[dtype] if dtype == 1 else FIT_TOL[0])
    vol.destroy()


def test_fitness_degenerate_inputs():
    rf = _rf()
    dims, vs, mu = (16, 16, 16), 0.05, 0.15
    vol = rf.Volume(dims, vs, mu)
    pst = _dev(S.sample_pst(33, 1))
    one = np.ones(6, np.float32)
    # empty (all-unobserved) volume: nothing can be sampled -> n = 0, rho = exp(-1) under F2
    pts = np.concatenate([np.random.default_rng(0).uniform(0.2, 0.6, (50, 3)), np.ones((50, 1))], 1).astype(np.float32)
    fit, cnt = vol.eval_particles(_dev(pts), pst, IDENT, one * 0.01)
    assert np.all(cnt.cpu().numpy() == 0) and np.allclose(fit.cpu().numpy(), math.exp(-1.0), rtol=1e-6)
    # every point masked out -> M_O = 0 -> rho = 0 (A22)
    pts[:, 3] = 0
    fit, cnt = vol.eval_particles(_dev(pts), pst, IDENT, one * 0.01)
    assert np.all(cnt.cpu().numpy() == 0) and np.all(fit.cpu().numpy() == 0)
    # invalid arguments are reported, not executed
    with pytest.raises(rf.RFError):
        vol.eval_particles(_dev(pts)[:0], pst, IDENT, one)
    with pytest.raises(rf.RFError):
        rf.Volume((0, 4, 4), 0.01, 0.04)
    with pytest.raises(rf.RFError):
        rf.Volume((8, 8, 8), 0.05, 0.01)                 # trunc < voxel_size
    vol.destroy()


# ---------------------------------------------------------------------------------- a0-a5 tracking
def _track_world():
    dims, vs, mu = (128, 128, 128), 0.02, 0.08
    scene = S.make_scene(4242, extent=2.56, inset=mu + 2 * vs, n_spheres=4, n_boxes=4, clearance=0.3)
    g = orc.make_grid(dims, vs, mu)
    w, h = 160, 120
    K = np.array([142.5, 142.5, 80.0, 60.0], dtype=np.float32)
    centre = 0.5 * (scene.room_lo + scene.room_hi)
    rng = np.random.Generator(np.random.Philox(77))
    pos = S.random_free_position(rng, scene, 0.35)
    T_prev = S.look_at(pos, centre + np.array([0.2, -0.1, -0.3])).astype(np.float32)
    F, W = orc.empty_volume(dims)
    for i in range(4):
        Ti = S.compose_delta(T_prev.astype(np.float64), [0, 0, 1], np.radians(-1.0 * (3 - i)), [0.01 * (i - 3), 0, 0])
        d = S.add_noise(S.raycast_depth(scene, Ti, K, w, h), 500 + i, sigma_rel=0.005)
        orc.integrate(g, F, W, d, K, Ti.astype(np.float32), nthreads=8)
    T_true = S.compose_delta(T_prev.astype(np.float64), [0.3, 0.5, 0.8], np.radians(10.0), [0.04, -0.03, 0.03])
    depth = S.add_noise(S.raycast_depth(scene, T_true, K, w, h), 600, sigma_rel=0.005, dropout=0.02)
    psts = [S.sample_pst(n, 700 + i) for i, n in enumerate((1024, 3072, 10240))]
    return dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true


def _oracle_iteration(g, F, W, depth, K, pst, stride, T32, Tprev32, r32, empty_run, variant=0, mode=0):
    """One PFO iteration composed from the pinned oracle primitives (O3, O6, O5, O7) on float32 state."""
    h, w = depth.shape
    pts = orc.backproject(depth, K, stride)
    if variant & orc.VAR_NO_OVERLAP:
        keep = (pts[:, 3] != 0).astype(np.float64)
        M_O = int(keep.sum())
    else:
        keep, M_O = orc.overlap_mask(pts, T32.astype(np.float64), Tprev32.astype(np.float64), K, w, h)
    p32 = pts.astype(np.float32)
    p32[:, 3] = keep
    cand = np.concatenate([np.zeros((1, 6), np.float32), pst], 0)          # candidate 0 = the centre (A14)
    ev = orc.eval_particles(g, F, W, p32, cand, T32, r32, mode=mode, nthreads=8)
    up = orc.swarm_update(ev["rho"], pst, T32.astype(np.float64), r32.astype(np.float64), empty_run, variant=variant)
    return ev, up, M_O


@pytest.mark.parametrize("dtype", [0, 1])
def test_pfo_iteration_parity_teacher_forced(dtype):
    """Per-iteration parity (A20, A21): for every iteration k both sides start from the SAME float32 state
    (the oracle's own state after k-1 iterations, rounded) and run exactly one iteration on level (k-1) mod 3."""
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    if dtype == 1:
        F = F.astype(np.float16).astype(np.float32)
    vol = rf.Volume(dims, vs, mu, dtype=dtype)
    vol.upload(F, W)
    strides = (2, 4, 8)
    dp = [_dev(p) for p in psts]
    dd = _dev(depth)
    tol = FIT_TOL[dtype]
    ref = orc.pfo_track(g, F, W, depth, K, psts, strides, 12, T_prev, T_prev, r0=np.full(6, 0.06), early_stop=False, nthreads=8)
    T32, r32 = T_prev.copy(), np.full(6, 0.06, dtype=np.float32)
    n_nonempty = 0
    for k in range(1, 13):
        l = (k - 1) % 3
        # a single-iteration call starts its own empty-run count at 0 on both sides; the "two empties in a row"
        # stop rule is covered by the free-run and no-usable-points tests
        ev, up, M_O = _oracle_iteration(g, F, W, depth, K, psts[l], strides[l], T32, T_prev, r32, 0)
        got = vol.pfo_track(dd, K, dp, strides, 1, T32, T_prev, r0=r32, flags=rf.RF_TRACK_NO_EARLY_STOP, want_trace=True,
                            start_iter=k - 1)
        gt = got["trace"][0]
        assert gt.level == l and gt.M_O == M_O, k
        assert abs(gt.rho_ref - up.rho_ref) <= tol * up.rho_ref, k
        assert abs(gt.rho_max - up.rho_max) <= tol * up.rho_max, k
        # candidates within tol of the threshold may legitimately flip in or out of the APS
        near = int(np.sum(np.abs(ev["rho"][1:] - up.rho_ref) <= 2 * tol * up.rho_ref))
        assert abs(gt.n_aps - up.n_aps) <= near, (k, gt.n_aps, up.n_aps, near)
        if up.n_aps - near > 0:
            n_nonempty += 1
            ds_o, ds_g = np.array(up.delta_star[:]), np.array(gt.delta_star[:])
            # A20: delta* is continuous in the fitness values; an error eps = tol*rho on every rho_j moves it by
            # at most 2 eps N_aps max|delta_j - delta*| / sum(omega) <= 4 eps N_aps max(r) / sum(omega)
            bound = 4 * tol * up.rho_max * max(r32) * (up.n_aps + near) / up.sum_omega + 1e-7
            assert np.max(np.abs(ds_g - ds_o)) <= bound, (k, np.max(np.abs(ds_g - ds_o)), bound)
            assert abs(gt.rho_tilde - up.rho_tilde) <= 4 * tol * up.rho_max * (up.n_aps + near) / up.sum_omega * (up.rho_max - up.rho_ref) + 2 * tol
            nv = np.linalg.norm(ds_o)
            rb = 0.9 * ((1 - up.rho_tilde) * 2 * np.sqrt(6) * bound / max(nv, 1e-12) + abs(gt.rho_tilde - up.rho_tilde)) + 1e-7
            assert np.max(np.abs(np.array(gt.r[:]) - np.array(up.r_new[:]))) <= rb, (k, rb)
            assert np.max(np.abs(np.array(gt.pose[:]) - np.array(up.T_new[:]))) <= 4 * bound * (1 + np.max(np.abs(T32))) + 1e-6, k
            assert gt.empty_run == 0
        elif up.n_aps == 0 and gt.n_aps == 0:
            assert np.allclose(np.array(gt.pose[:]).reshape(3, 4), T32.astype(np.float64), atol=0)      # pose unchanged
            assert np.allclose(gt.r[:], up.r_new[:], rtol=0, atol=4 * tol)
            assert gt.empty_run == up.empty_run and gt.stop == up.stop
        if k == 1:
            assert np.allclose(got["r1"], np.array(up.r_new[:]), atol=max(1e-6, 10 * tol * max(r32)) if up.n_aps else 4 * tol)
        # next teacher state: the oracle's free-running state after k iterations, rounded to float32
        row = ref["trace"][k - 1]
        T32 = np.array(row.pose[:], dtype=np.float32).reshape(3, 4)
        r32 = np.array(row.r[:], dtype=np.float32)
    assert n_nonempty >= 3                                   # the comparison above was exercised
    vol.destroy()


@pytest.mark.parametrize("early", [False, True])
def test_pfo_track_free_run_ends_where_the_oracle_ends(early):
    """Free-running 20 iterations.  Within a frame the two trajectories may drift apart at APS-threshold flips
    (A20, A21), so this is a sanity check on the outcome, not the parity gate (that is the test above)."""
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    vol = rf.Volume(dims, vs, mu)
    vol.upload(F, W)
    strides = (2, 4, 8)
    flags = 0 if early else rf.RF_TRACK_NO_EARLY_STOP
    got = vol.pfo_track(_dev(depth), K, [_dev(p) for p in psts], strides, 20, T_prev, T_prev, r0=None, flags=flags,
                        want_trace=True)
    ref = orc.pfo_track(g, F, W, depth, K, psts, strides, 20, T_prev, T_prev, r0=None, early_stop=early, nthreads=8)
    if not early:
        assert got["iters_run"] == ref["iters_run"] == 20
    # iteration 1 starts from identical state: it must agree tightly
    g1, o1 = got["trace"][0], ref["trace"][0]
    assert g1.M_O == o1.M_O and abs(g1.rho_ref - o1.rho_ref) <= 1e-5 * o1.rho_ref and abs(g1.n_aps - o1.n_aps) <= 2
    e0 = np.linalg.norm(T_prev[:, 3] - T_true[:, 3])
    e_gpu = np.linalg.norm(got["pose"][:, 3] - T_true[:, 3])
    e_orc = np.linalg.norm(ref["pose"][:, 3] - T_true[:, 3])
    assert e_gpu < 0.3 * e0 and e_orc < 0.3 * e0              # both recover the 10 deg / 6 cm offset
    assert abs(e_gpu - e_orc) < 0.01
    assert abs(got["trace"][-1].rho_ref - ref["trace"][-1].rho_ref) < 0.01
    vol.destroy()


def test_pfo_track_second_frame_uses_r1_and_host_depth():
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    vol = rf.Volume(dims, vs, mu)
    vol.upload(F, W)
    dp = [_dev(p) for p in psts]
    r0 = np.array([0.03, 0.04, 0.05, 0.06, 0.03, 0.02], dtype=np.float32)
    got = vol.pfo_track(depth, K, dp, (2, 4, 8), 6, T_prev, T_prev, r0=r0, want_trace=True)       # host depth
    ref = orc.pfo_track(g, F, W, depth, K, psts, (2, 4, 8), 6, T_prev, T_prev, r0=r0.astype(np.float64), nthreads=8)
    # iteration 1 starts from identical state (the caller's r0, host depth): tight; r1 is that iteration's r
    g1, o1 = got["trace"][0], ref["trace"][0]
    assert g1.M_O == o1.M_O and np.allclose(g1.rho_ref, o1.rho_ref, rtol=3e-5) and abs(g1.n_aps - o1.n_aps) <= 2
    assert np.max(np.abs(np.array(g1.pose[:]) - np.array(o1.pose[:]))) <= 2e-4
    assert np.allclose(got["r1"], ref["r1"], atol=5e-4) and np.allclose(got["r1"], list(g1.r), atol=1e-7)
    # the free run of six iterations may drift at advantage-set threshold flips (A20, A21): loose bound on where it ends
    assert np.max(np.abs(got["pose"].astype(np.float64) - ref["pose"])) <= 1e-2
    vol.destroy()


def test_pfo_track_no_usable_points():
    rf = _rf()
    vol = rf.Volume((32, 32, 32), 0.05, 0.15)
    depth = np.zeros((48, 64), np.float32)               # every pixel invalid
    psts = [_dev(S.sample_pst(n, 1 + i)) for i, n in enumerate((64, 128, 256))]
    K = np.array([50, 50, 31.5, 23.5], np.float32)
    got = vol.pfo_track(_dev(depth), K, psts, (2, 4, 8), 5, IDENT, IDENT)
    assert got["status"] & rf.RF_TRACK_NO_POINTS
    assert np.array_equal(got["pose"], IDENT) and got["evals"] == 0
    assert got["iters_run"] == 2                          # APS empty twice in a row
    with pytest.raises(rf.RFError):
        vol.pfo_track(_dev(depth), K, psts, (2, 4, 8), 0, IDENT, IDENT)
    vol.destroy()


def test_pfo_track_launch_modes_are_bit_identical_and_graph_replays():
    """The frame loop as a CUDA graph with programmatic dependent launch, as a graph without it, and launched
    kernel by kernel must give the SAME bits (fixed-shape reductions, integer accumulation); replaying the cached
    graph on new inputs must track those inputs, and early stop inside a replayed graph must still work."""
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    vol = rf.Volume(dims, vs, mu, dtype=1)
    vol.upload(F.astype(np.float16).astype(np.float32), W)
    dp = [_dev(p) for p in psts]
    dd = _dev(depth)
    r0 = np.full(6, 0.06, dtype=np.float32)
    runs = {}
    for name, fl in (("graph+pdl", 0), ("graph", rf.RF_TRACK_NO_PDL), ("direct", rf.RF_TRACK_NO_GRAPH | rf.RF_TRACK_NO_PDL),
                     ("direct+pdl", rf.RF_TRACK_NO_GRAPH)):
        runs[name] = vol.pfo_track(dd, K, dp, (2, 4, 8), 9, T_prev, T_prev, r0=r0, flags=fl | rf.RF_TRACK_NO_EARLY_STOP,
                                   want_trace=True)
    base = runs["direct"]
    for name, out in runs.items():
        assert out["iters_run"] == 9 and out["evals"] == base["evals"], name
        assert np.array_equal(out["pose"], base["pose"]) and np.array_equal(out["r1"], base["r1"]), name
        for a, b in zip(out["trace"], base["trace"]):
            assert bytes(a) == bytes(b), name
    # replay of the cached graph with different inputs (same shapes): must equal a direct launch on those inputs
    T2 = S.compose_delta(T_prev.astype(np.float64), [0, 1, 0], np.radians(2.0), [0.01, 0.0, -0.01]).astype(np.float32)
    r2 = np.array([0.02, 0.03, 0.04, 0.05, 0.06, 0.07], dtype=np.float32)
    a = vol.pfo_track(dd, K, dp, (2, 4, 8), 9, T2, T_prev, r0=r2, flags=rf.RF_TRACK_NO_EARLY_STOP, want_trace=True)
    b = vol.pfo_track(dd, K, dp, (2, 4, 8), 9, T2, T_prev, r0=r2, flags=rf.RF_TRACK_NO_EARLY_STOP | rf.RF_TRACK_NO_GRAPH | rf.RF_TRACK_NO_PDL,
                      want_trace=True)
    assert np.array_equal(a["pose"], b["pose"]) and not np.array_equal(a["pose"], base["pose"])
    assert all(bytes(x) == bytes(y) for x, y in zip(a["trace"], b["trace"]))
    # early stop inside a graph: the remaining launches are no-ops
    c = vol.pfo_track(dd, K, dp, (2, 4, 8), 20, T_prev, T_prev, r0=np.full(6, 1e-4, dtype=np.float32), want_trace=True)
    d = vol.pfo_track(dd, K, dp, (2, 4, 8), 20, T_prev, T_prev, r0=np.full(6, 1e-4, dtype=np.float32), want_trace=True,
                      flags=rf.RF_TRACK_NO_GRAPH | rf.RF_TRACK_NO_PDL)
    assert c["iters_run"] == d["iters_run"] and c["status"] == d["status"] and np.array_equal(c["pose"], d["pose"])
    vol.destroy()


@pytest.mark.parametrize("name", ["no_overlap", "rescale_iso", "rescale_aniso", "eq14"])
def test_pfo_iteration_parity_ablation_variants(name):
    """The paper's ablations (Fig. 11, Table 2) through the same teacher-forced per-iteration
    gate as the default path (A20, A21)."""
    rf = _rf()
    gpu_flag, variant, mode = {"no_overlap": (rf.RF_TRACK_NO_OVERLAP, orc.VAR_NO_OVERLAP, 0),
                               "rescale_iso": (rf.RF_TRACK_RESCALE_ISO, orc.VAR_RESCALE_ISO, 0),
                               "rescale_aniso": (rf.RF_TRACK_RESCALE_ANISO, orc.VAR_RESCALE_ANISO, 0),
                               "eq14": (rf.RF_TRACK_MODE_EQ14, 0, 2)}[name]
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    # a previous pose that sees only part of the frame makes Eq. (19) and "No Overlap" differ
    T_old = S.compose_delta(T_prev.astype(np.float64), [0, 1, 0], np.radians(25.0), [0.0, 0.0, 0.0]).astype(np.float32)
    vol = rf.Volume(dims, vs, mu, dtype=0)
    vol.upload(F, W)
    strides = (2, 4, 8)
    dp = [_dev(p) for p in psts]
    dd = _dev(depth)
    ref = orc.pfo_track(g, F, W, depth, K, psts, strides, 6, T_prev, T_old, r0=np.full(6, 0.06), early_stop=False, nthreads=8,
                        variant=variant, mode=mode)
    T32, r32 = T_prev.copy(), np.full(6, 0.06, dtype=np.float32)
    checked = 0
    for k in range(1, 7):
        l = (k - 1) % 3
        ev, up, M_O = _oracle_iteration(g, F, W, depth, K, psts[l], strides[l], T32, T_old, r32, 0, variant, mode)
        got = vol.pfo_track(dd, K, dp, strides, 1, T32, T_old, r0=r32, flags=rf.RF_TRACK_NO_EARLY_STOP | gpu_flag,
                            want_trace=True, start_iter=k - 1)
        gt = got["trace"][0]
        # Eq. (14) is Eq. (20) to the power |O|: the relative tolerance on rho scales with |O|
        tol = 1e-5 * (M_O if mode == 2 else 1)
        assert gt.M_O == M_O, (k, gt.M_O, M_O)
        assert abs(gt.rho_ref - up.rho_ref) <= tol * up.rho_ref, k
        assert abs(gt.rho_max - up.rho_max) <= tol * up.rho_max, k
        near = int(np.sum(np.abs(ev["rho"][1:] - up.rho_ref) <= 2 * tol * up.rho_ref))
        assert abs(gt.n_aps - up.n_aps) <= near, (k, gt.n_aps, up.n_aps, near)
        if up.n_aps - near > 0 and mode != 2:
            bound = 4 * tol * up.rho_max * max(r32) * (up.n_aps + near) / up.sum_omega + 1e-7
            ds_o, ds_g = np.array(up.delta_star[:]), np.array(gt.delta_star[:])
            assert np.max(np.abs(ds_g - ds_o)) <= bound, (k, np.max(np.abs(ds_g - ds_o)), bound)
            nv = np.linalg.norm(ds_o)
            rb = 0.9 * (2 * np.sqrt(6) * bound / max(nv, 1e-12) + abs(gt.rho_tilde - up.rho_tilde)) + 1e-7
            assert np.max(np.abs(np.array(gt.r[:]) - np.array(up.r_new[:]))) <= rb, (k, rb)
            checked += 1
        elif mode == 2 and up.n_aps > 0:
            # weights omega span hundreds of orders of magnitude under Eq. (14): the best particle dominates
            assert gt.argmax == up.argmax or abs(gt.rho_max - up.rho_max) <= tol * up.rho_max
            assert np.max(np.abs(np.array(gt.pose[:]) - np.array(up.T_new[:]))) <= 1e-3
            checked += 1
        row = ref["trace"][k - 1]
        T32 = np.array(row.pose[:], dtype=np.float32).reshape(3, 4)
        r32 = np.array(row.r[:], dtype=np.float32)
    assert checked >= (1 if mode == 2 else 2)        # under Eq. (14) the advantage set empties after one step here
    if name == "no_overlap":
        full = orc.backproject(depth, K, strides[0])
        assert ref["trace"][0].M_O == int((full[:, 3] != 0).sum())
        assert orc.overlap_mask(full, T_prev.astype(np.float64), T_old.astype(np.float64), K, depth.shape[1], depth.shape[0])[1] < ref["trace"][0].M_O
    vol.destroy()


def test_stage_frame_prefetch_equals_direct_host_depth():
    """rf_stage_frame + rf_pfo_track(depth_on_host = 2) + rf_integrate_ex(depth_on_host = 2) must give the bits of the
    plain host-depth calls; slots are consumed in order; a third pending frame and an empty queue are errors."""
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    depth2 = np.ascontiguousarray(depth[::-1, :].copy())                     # a second, different frame
    dp = [_dev(p) for p in psts]
    r0 = np.full(6, 0.05, dtype=np.float32)
    outs = {}
    for mode in ("direct", "prefetch"):
        vol = rf.Volume(dims, vs, mu)
        vol.upload(F, W)
        res = []
        if mode == "prefetch":
            pins = [torch.from_numpy(depth).pin_memory(), torch.from_numpy(depth2).pin_memory()]
            vol.stage_frame(pins[0]); vol.stage_frame(pins[1])
            with pytest.raises(rf.RFError):
                vol.stage_frame(pins[0])                                    # both slots pending
        for i, d in enumerate((depth, depth2)):
            src = d if mode == "direct" else tuple(d.shape)
            o = vol.pfo_track(src, K, dp, (2, 4, 8), 4, T_prev, T_prev, r0=r0, flags=rf.RF_TRACK_NO_EARLY_STOP)
            if mode == "direct":
                vol.integrate(d, K, o["pose"])
            else:
                vol.integrate(None, K, o["pose"], staged_shape=d.shape)
            res.append(o)
        if mode == "prefetch":
            with pytest.raises(rf.RFError):
                vol.pfo_track(tuple(depth.shape), K, dp, (2, 4, 8), 1, T_prev, T_prev, r0=r0)     # nothing pending
        outs[mode] = (res, vol.download())
        vol.destroy()
    for a, b in zip(outs["direct"][0], outs["prefetch"][0]):
        assert np.array_equal(a["pose"], b["pose"]) and a["evals"] == b["evals"]
    assert not np.array_equal(outs["direct"][0][0]["pose"], outs["direct"][0][1]["pose"])
    assert all(np.array_equal(x, y) for x, y in zip(outs["direct"][1], outs["prefetch"][1]))


def test_pfo_track_ragged_pst_sizes_and_strides():
    """Template sizes that are not multiples of the CTA width (128) or of the update cluster's stride, strides that do
    not divide the image: iteration 1 against the oracle (identical start state), and graph == kernel-by-kernel."""
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    sizes = (777, 1500, 2049)
    ps = [S.sample_pst(n, 900 + i) for i, n in enumerate(sizes)]
    strides = (3, 5, 7)
    vol = rf.Volume(dims, vs, mu)
    vol.upload(F, W)
    dp = [_dev(p) for p in ps]
    r0 = np.full(6, 0.05, dtype=np.float32)
    a = vol.pfo_track(_dev(depth), K, dp, strides, 7, T_prev, T_prev, r0=r0, flags=rf.RF_TRACK_NO_EARLY_STOP, want_trace=True)
    b = vol.pfo_track(_dev(depth), K, dp, strides, 7, T_prev, T_prev, r0=r0,
                      flags=rf.RF_TRACK_NO_EARLY_STOP | rf.RF_TRACK_NO_GRAPH | rf.RF_TRACK_NO_PDL, want_trace=True)
    assert np.array_equal(a["pose"], b["pose"]) and all(bytes(x) == bytes(y) for x, y in zip(a["trace"], b["trace"]))
    ref = orc.pfo_track(g, F, W, depth, K, ps, strides, 7, T_prev, T_prev, r0=r0.astype(np.float64), early_stop=False, nthreads=8)
    g1, o1 = a["trace"][0], ref["trace"][0]
    h, w = depth.shape
    assert g1.M_O == o1.M_O <= orc.lattice_count(w, 3) * orc.lattice_count(h, 3)
    assert abs(g1.rho_ref - o1.rho_ref) <= 1e-5 * o1.rho_ref and abs(g1.rho_max - o1.rho_max) <= 1e-5 * o1.rho_max
    assert abs(g1.n_aps - o1.n_aps) <= 2
    if o1.n_aps > 2:
        assert np.max(np.abs(np.array(g1.pose[:]) - np.array(o1.pose[:]))) <= 1e-4
    assert a["evals"] == sum(int(t.M_O) * (sizes[i % 3] + 1) for i, t in enumerate(a["trace"]))
    vol.destroy()


# ---------------------------------------------------------------------------------- read-out (rf_raycast vs O9)
def _raycast_compare(vol, g, F, W, K, w, h, pose, step, z_max):
    d, n = vol.raycast(K, w, h, pose, step, z_max, want_normals=True)
    d, n = d.cpu().numpy(), n.cpu().numpy()
    od, on, frag = orc.raycast(g, F, W, K, w, h, pose, step, z_max, nthreads=8)
    solid = frag == 0
    hit = od > 0
    # pixels the oracle does not flag take the same hit / no-hit decision and the same interval
    assert np.array_equal(d[solid] > 0, hit[solid])
    m = solid & hit
    if m.any():
        # fp32 blend of exact corner values: |d psi| ~ 2e-7, crossing denominator >= 1e-3 (else flagged), step <= 0.1 m
        assert np.max(np.abs(d[m] - od[m])) <= 1e-5
    fin = np.isfinite(on).all(-1)
    assert np.array_equal(np.isfinite(n).all(-1)[m], fin[m])
    mm = m & fin
    if mm.any():
        assert np.max(np.abs(n[mm] - on[mm])) <= 1e-4
    assert np.all(np.isnan(n[solid & ~hit]))
    # flagged pixels: whatever interval the kernel took, the answer is a depth of the march or 0
    assert np.all((d[~solid] == 0) | ((d[~solid] > 0) & (d[~solid] <= z_max)))
    return hit.mean(), frag.mean(), fin[m].mean() if m.any() else 0.0


@pytest.mark.parametrize("dtype", [0, 1])
def test_raycast_parity_observed_scene(dtype):
    """128^3 volume fused from 4 noisy frames (oracle-built): two views, one with an image size that is not a multiple of
    the 16x16 pixel tile; fp16 volumes hold the fp16-rounded values on both sides."""
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    if dtype == 1:
        F = F.astype(np.float16).astype(np.float32)
    vol = rf.Volume(dims, vs, mu, dtype=dtype)
    vol.upload(F, W)
    step, z_max = float(np.float32(0.5 * mu)), 4.0
    hit, frag, fin = _raycast_compare(vol, g, F, W, K, 160, 120, T_prev, step, z_max)
    assert hit > 0.5 and frag < 0.05 and fin > 0.8
    K2 = np.array([150.0, 148.0, 86.0, 65.0], dtype=np.float32)
    hit, frag, fin = _raycast_compare(vol, g, F, W, K2, 173, 131, T_true.astype(np.float32), float(np.float32(0.3 * mu)), 3.0)
    assert hit > 0.3 and frag < 0.05
    vol.destroy()


def test_raycast_ragged_volume_outside_camera_and_empty_cases():
    rf = _rf()
    dims, vs, mu = (70, 66, 50), 0.03, 0.09
    scene, K, w, h, poses, frames = _small_world(dims, vs, mu)
    g = orc.make_grid(dims, vs, mu)
    F, W = orc.empty_volume(dims)
    for T, d in zip(poses, frames):
        orc.integrate(g, F, W, d, K, T, half_storage=True, nthreads=8)
    vol = rf.Volume(dims, vs, mu, dtype=rf.RF_F16_W8)
    vol.upload(F, W)
    step = float(np.float32(0.04))
    hit, frag, _ = _raycast_compare(vol, g, F, W, K, w, h, poses[0], step, 5.0)
    assert hit > 0.2
    # a camera outside the grid looking in, and one looking away
    back = poses[0].astype(np.float64).copy()
    back[:, 3] -= 1.5 * back[:, 2]
    hit2, _, _ = _raycast_compare(vol, g, F, W, K, w, h, back.astype(np.float32), step, 6.0)
    assert hit2 > 0.02
    away = back.copy()
    away[:, :3] = away[:, :3] @ np.diag([-1.0, 1.0, -1.0])
    d, n = vol.raycast(K, w, h, away.astype(np.float32), step, 6.0, want_normals=True)
    assert float(d.abs().max()) == 0.0 and bool(n.isnan().all())
    # z_max shorter than one step: no samples; depth only (normals NULL)
    d, n = vol.raycast(K, w, h, poses[0], step, 0.01)
    assert n is None and float(d.abs().max()) == 0.0
    # an empty volume has no surface; a reset after the atlas exists must be seen by the next read-out
    vol.reset()
    d, _ = vol.raycast(K, w, h, poses[0], step, 5.0)
    assert float(d.abs().max()) == 0.0
    with pytest.raises(rf.RFError):
        vol.raycast(K, w, h, poses[0], 0.0, 5.0)
    vol.destroy()


def test_track_integrate_is_track_then_integrate_bit_for_bit():
    """rf_track_integrate == rf_pfo_track + rf_integrate at the returned pose (device depth and host depth), and the gate
    holds a frame back without touching the volume."""
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    dp = [_dev(p) for p in psts]
    r0 = np.full(6, 0.05, dtype=np.float32)
    res = {}
    for name in ("two_calls", "fused_dev", "fused_host", "gated"):
        vol = rf.Volume(dims, vs, mu, dtype=rf.RF_F16_W8)
        vol.upload(F, W)
        if name == "two_calls":
            out = vol.pfo_track(_dev(depth), K, dp, (4, 8, 16), 6, T_prev, T_prev, r0=r0)
            assert out["integrated"] is False
            vol.integrate(_dev(depth), K, out["pose"])
        elif name == "fused_dev":
            out = vol.track_integrate(_dev(depth), K, dp, (4, 8, 16), 6, T_prev, T_prev, r0=r0,
                                      gate=(out["pose"][:, 3], 0.01))
            assert out["integrated"] is True
        elif name == "fused_host":
            out = vol.track_integrate(depth, K, dp, (4, 8, 16), 6, T_prev, T_prev, r0=r0)
            assert out["integrated"] is True
        else:
            out = vol.track_integrate(_dev(depth), K, dp, (4, 8, 16), 6, T_prev, T_prev, r0=r0,
                                      gate=(out["pose"][:, 3] + np.array([0.5, 0, 0], dtype=np.float32), 0.1))
            assert out["integrated"] is False
        res[name] = (out["pose"].copy(), out["r1"].copy(), vol.last_updated() if name != "gated" else 0) + vol.download()
        vol.destroy()
    for name in ("fused_dev", "fused_host"):
        assert np.array_equal(res[name][0], res["two_calls"][0]) and np.array_equal(res[name][1], res["two_calls"][1])
        assert res[name][2] == res["two_calls"][2] > 0
        assert np.array_equal(res[name][3], res["two_calls"][3], equal_nan=True) and np.array_equal(res[name][4], res["two_calls"][4])
    assert np.array_equal(res["gated"][0], res["two_calls"][0])
    Fq = F.astype(np.float16).astype(np.float32)
    assert np.array_equal(res["gated"][4], W) and np.array_equal(res["gated"][3][W > 0], Fq[W > 0])

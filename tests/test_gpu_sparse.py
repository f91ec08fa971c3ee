"""Sparse volumes (rf_volume_opts.pool_bricks > 0; SURVEY 8(f)-3 "sparse/bricked allocation for volumes beyond 1024^3").

A sparse volume stores only the bricks an integration has swept; everything it computes must be what a dense volume
computes.  (1) Same dims and origin, dense and sparse side by side: the fused volume, the fitness of a swarm, a whole
tracked frame and the fused result after it are bit-identical (same kernels, same arithmetic; only the place a brick is
stored differs).  (2) A 2048^3 logical grid (8.6 G voxels: it could not be stored densely with its atlas) holding the same
small world at voxel offset 512: integration against the oracle through the usual gate (tests/gates.py), fitness against the
oracle sampled on the box around the world.  (3) A pool that is too small drops bricks and says so.  (4) Upload gives the bricks
with an observed voxel a slot (and fails loudly if the pool is too small); the read-outs of an empty sparse volume find nothing."""
import numpy as np
import pytest

import oracle as orc
import rf_synth as S
from gates import check_integration
from test_gpu_parity import _check_fitness, _dev, _rf, _small_world

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dtype", [0, 1])
def test_sparse_volume_is_bit_identical_to_dense(dtype):
    rf = _rf()
    dims, vs, mu = (70, 66, 50), 0.03, 0.09
    scene, K, w, h, poses, frames = _small_world(dims, vs, mu, n_frames=4)
    nbricks = 9 * 9 * 7
    dense = rf.Volume(dims, vs, mu, dtype=dtype)
    sparse = rf.Volume(dims, vs, mu, dtype=dtype, pool_bricks=nbricks)
    for T, d in zip(poses[:3], frames[:3]):
        dense.integrate(_dev(d), K, T)
        sparse.integrate(_dev(d), K, T)
        assert dense.last_updated() == sparse.last_updated() > 1000
    st = sparse.pool_stats()
    assert 0 < st["allocated"] < nbricks and st["capacity"] == nbricks and st["dropped_last"] == 0
    Fd, Wd = dense.download()
    Fs, Ws = sparse.download()
    assert np.array_equal(Wd, Ws) and np.array_equal(Fd, Fs) and (Wd > 0).mean() > 0.03
    bt, bw = sparse.download_box((8, 16, 5), (40, 33, 30))                      # a box that is not brick-aligned
    ref_t = Fd.reshape(dims[2], dims[1], dims[0])[5:35, 16:49, 8:48]
    ref_w = Wd.reshape(dims[2], dims[1], dims[0])[5:35, 16:49, 8:48]
    assert np.array_equal(bt.cpu().numpy(), ref_t) and np.array_equal(bw.cpu().numpy(), ref_w)
    dt, dw = dense.download_box((8, 16, 5), (40, 33, 30))
    assert np.array_equal(dt.cpu().numpy(), ref_t) and np.array_equal(dw.cpu().numpy(), ref_w)
    # fitness of a swarm around the last pose (several CTAs, points that leave the grid and the observed region)
    depth = _dev(frames[3])
    pst = S.sample_pst(1500, 4242)
    r = np.array([0.03, 0.03, 0.03, 0.05, 0.05, 0.05], dtype=np.float32)
    pts = dense.backproject(depth, K, 2)
    fd, cd = dense.eval_particles(pts, _dev(pst), poses[3], r)
    fs, cs = sparse.eval_particles(pts, _dev(pst), poses[3], r)
    assert torch.equal(fd, fs) and torch.equal(cd, cs) and int(cd.max()) > 500
    # a whole tracked frame and its fusion
    psts = [_dev(S.sample_pst(n, 900 + i)) for i, n in enumerate((256, 512, 1024))]
    rd = dense.track_integrate(depth, K, psts, (2, 4, 8), 12, poses[2], poses[2])
    rs = sparse.track_integrate(depth, K, psts, (2, 4, 8), 12, poses[2], poses[2])
    assert np.array_equal(rd["pose"], rs["pose"]) and rd["iters_run"] == rs["iters_run"] and rd["evals"] == rs["evals"]
    Fd, Wd = dense.download()
    Fs, Ws = sparse.download()
    assert np.array_equal(Wd, Ws) and np.array_equal(Fd, Fs)
    # the read-outs and the Gauss-Newton tracker go through the same indirection
    zd, nd = dense.raycast(K, w, h, poses[3], 0.02, 3.0, want_normals=True)
    zs, ns = sparse.raycast(K, w, h, poses[3], 0.02, 3.0, want_normals=True)
    assert torch.equal(zd, zs) and torch.equal(torch.nan_to_num(nd, nan=7.0), torch.nan_to_num(ns, nan=7.0)) and int((zd > 0).sum()) > 2000
    pd, ed = dense.extract_surface_points()
    ps, es = sparse.extract_surface_points()
    od, os_ = torch.argsort(ed), torch.argsort(es)
    assert torch.equal(ed[od], es[os_]) and torch.equal(pd[od], ps[os_]) and ed.numel() > 500
    T0 = S.compose_delta(np.asarray(poses[3], dtype=np.float64), [0.2, 0.9, -0.1], np.radians(1.0), [0.01, -0.005, 0.008])
    gd, gs = dense.gn_track(pts, T0, 5), sparse.gn_track(pts, T0, 5)
    assert gd["iters_run"] == gs["iters_run"] == 5 and np.array_equal(gd["pose"], gs["pose"]) and gd["rows"][0].n > 500
    assert all(a.n == b.n and a.cost == b.cost and list(a.A) == list(b.A) for a, b in zip(gd["rows"], gs["rows"]))
    gz = sparse.gn_track_noalloc(pts, T0, 5)
    assert np.array_equal(gz["pose"], gd["pose"])
    # reset empties the pool; the volume can be filled again
    sparse.reset()
    assert sparse.pool_stats()["allocated"] == 0
    Fs, Ws = sparse.download()
    assert not Ws.any() and np.all(Fs == 1.0)
    sparse.integrate(_dev(frames[0]), K, poses[0])
    dense.reset()
    dense.integrate(_dev(frames[0]), K, poses[0])
    assert all(np.array_equal(a, b) for a, b in zip(dense.download(), sparse.download()))
    dense.destroy()
    sparse.destroy()


def test_sparse_logical_grid_of_2048_cubed_against_the_oracle():
    rf = _rf()
    dims, vs, mu = (70, 66, 50), 0.03125, 0.09375                    # vs = 2^-5: the offset grid has exactly the same voxel centres
    scene, K, w, h, poses, frames = _small_world(dims, vs, mu, n_frames=4)
    OFF = 512                                                        # voxels (64 bricks) between the grid's corner and the world's
    big = (2048, 2048, 2048)
    vol = rf.Volume(big, vs, mu, dtype=rf.RF_F16_W8, origin=(-OFF * vs,) * 3, pool_bricks=4096)
    g = orc.make_grid(dims, vs, mu)                                  # the oracle works on the box around the world, origin 0
    F, W = orc.empty_volume(dims)
    frag_all = np.zeros(F.size, dtype=np.uint8)
    d_prev = None
    for i, (T, d) in enumerate(zip(poses[:3], frames[:3])):
        Wprev = W.copy()
        frag = np.zeros(F.size, dtype=np.uint8)
        orc.integrate(g, F, W, d, K, T, half_storage=True, nthreads=8, fragile=frag)
        frag_all |= frag
        vol.integrate(_dev(d), K, T)
        bt, bw = vol.download_box((OFF, OFF, OFF), dims)
        Ft, Wt = bt.cpu().numpy().reshape(-1), bw.cpu().numpy().reshape(-1)
        ff, _, d_prev = check_integration(Ft, Wt, F, W, Wprev, frag_all, True, vs, mu, tag=i, d_prev=d_prev, frames=i + 1)
        assert ff < 0.03
    st = vol.pool_stats()
    assert 100 < st["allocated"] <= 9 * 9 * 7 + 400 and st["dropped_last"] == 0          # the world's bricks and a rim, of 16.7 M
    assert (W > 0).mean() > 0.03
    # nothing is observed outside the box around the world
    rim_t, rim_w = vol.download_box((OFF - 16, OFF - 16, OFF - 16), (16, 98, 82))
    assert not rim_w.any().item() and bool((rim_t == 1.0).all())
    # fitness: the oracle samples the values the CUDA path holds in the box (outside it nothing is observed on either side)
    depth = _dev(frames[3])
    pts = vol.backproject(depth, K, 2)
    pst = S.sample_pst(1024, 777)
    r = np.array([0.03, 0.03, 0.03, 0.05, 0.05, 0.05], dtype=np.float32)
    fit, cnt = vol.eval_particles(pts, _dev(pst), poses[3], r)
    ref = orc.eval_particles(g, Ft, Wt, pts.cpu().numpy(), pst, poses[3], r, nthreads=8)
    assert ref["n"].max() > 500
    _check_fitness(fit, cnt, ref, 2e-3)
    vol.destroy()


def test_sparse_pool_too_small_drops_bricks_and_reports_them():
    rf = _rf()
    dims, vs, mu = (70, 66, 50), 0.03, 0.09
    scene, K, w, h, poses, frames = _small_world(dims, vs, mu)
    dense = rf.Volume(dims, vs, mu, dtype=rf.RF_F16_W8)
    small = rf.Volume(dims, vs, mu, dtype=rf.RF_F16_W8, pool_bricks=60)
    dense.integrate(_dev(frames[0]), K, poses[0])
    small.integrate(_dev(frames[0]), K, poses[0])
    st = small.pool_stats()
    assert st["allocated"] == 60 and st["dropped_last"] > 0
    Fd, Wd = dense.download()
    Fs, Ws = small.download()
    kept = Ws > 0
    assert 0 < kept.sum() < (Wd > 0).sum()                           # some of the frame was fused, not all of it
    assert np.array_equal(Ws[kept], Wd[kept]) and np.array_equal(Fs[kept], Fd[kept])      # and what was fused is right
    assert small.last_updated() == int(kept.sum())
    dense.destroy()
    small.destroy()


def test_sparse_upload_roundtrip_and_empty_read_outs():
    rf = _rf()
    dims, vs, mu = (64, 64, 64), 0.03, 0.09
    vol = rf.Volume(dims, vs, mu, dtype=rf.RF_F16_W8, pool_bricks=128)
    K = np.array([80.0, 80.0, 47.5, 35.5], dtype=np.float32)
    I = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0]], dtype=np.float32)
    # an empty sparse volume: every read-out finds nothing
    z, _ = vol.raycast(K, 96, 72, I, 0.01, 2.0)
    assert not z.any().item() and vol.extract_surface_points()[0].shape[0] == 0
    assert vol.gn_track(torch.ones((16, 4), device="cuda"), I, 2)["rows"][0].n == 0
    # upload: the bricks with an observed voxel get slots (here a slab of 2 x 8 x 3 bricks and one lone voxel)
    rng = np.random.default_rng(11)
    W = np.zeros((64, 64, 64), dtype=np.float32)                      # [z, y, x]
    W[10:30, :, 3:14] = rng.integers(0, 4, size=(20, 64, 11))
    W[50, 50, 50] = 7
    F = rng.uniform(-1, 1, size=W.shape).astype(np.float16).astype(np.float32)
    vol.upload(F.reshape(-1), W.reshape(-1))
    st = vol.pool_stats()
    assert st["allocated"] == 2 * 8 * 3 + 1 and st["dropped_last"] == 0
    Ft, Wt = vol.download()
    assert np.array_equal(Wt, W.reshape(-1)) and np.array_equal(Ft, np.where(W > 0, F, 1.0).reshape(-1))
    small = rf.Volume(dims, vs, mu, dtype=rf.RF_F16_W8, pool_bricks=16)
    with pytest.raises(rf.RFError, match="pool is too small"):
        small.upload(F.reshape(-1), W.reshape(-1))
    small.destroy()
    with pytest.raises(rf.RFError):
        rf.Volume((8192, 8192, 8192), vs, mu, pool_bricks=128)          # 2^30 logical bricks: beyond the 2^25 limit
    vol.destroy()

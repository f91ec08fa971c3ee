"""GPU parity of the options of the CUDA path that the main parity files do not reach: a non-zero volume origin
(fitness, integration, read-out), weight caps below 255 and the running average beyond the cap, invalid depth values,
the F1 normalisation inside the frame loop, the two-empties stop rule over a multi-iteration call, the five-argument
rf_volume_create, and argument errors.  Gates as in test_gpu_parity.py / tests/gates.py."""
import numpy as np
import pytest

import oracle as orc
import rf_synth as S
from gates import check_integration
from test_gpu_parity import FIT_TOL, _check_fitness, _dev, _oracle_iteration, _raycast_compare, _rf, _small_world, _track_world

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

ORIGIN = np.array([-1.3, 0.7, 2.1])


def _shift(T, o):
    T = np.array(T, dtype=np.float64).copy()
    T[:, 3] += o
    return T.astype(np.float32)


@pytest.mark.parametrize("dtype", [0, 1])
def test_nonzero_origin_integration_fitness_and_readout(dtype):
    """The whole world (grid origin and camera poses) moved by a vector with no binary32-friendly components: the same
    geometry relative to the grid, different numbers everywhere (rf_fitness.cu grid-space matrix, make_params, ray set-up)."""
    rf = _rf()
    dims, vs, mu = (70, 66, 50), 0.03, 0.09
    scene, K, w, h, poses, frames = _small_world(dims, vs, mu)
    g = orc.make_grid(dims, vs, mu, ORIGIN)
    o32 = np.array(g.origin[:], dtype=np.float64)                 # the origin both sides see (binary32)
    F, W = orc.empty_volume(dims)
    vol = rf.Volume(dims, vs, mu, dtype=dtype, origin=ORIGIN)
    for i, (T, d) in enumerate(zip(poses, frames)):
        Ts = _shift(T, o32)
        Fprev, Wprev = F.copy(), W.copy()
        frag = np.zeros(F.size, dtype=np.uint8)
        orc.integrate(g, F, W, d, K, Ts, half_storage=(dtype == 1), nthreads=8, fragile=frag)
        vol.upload(Fprev, Wprev)
        vol.integrate(_dev(d), K, Ts)
        Ft, Wt = vol.download()
        ff, _, _ = check_integration(Ft, Wt, F, W, Wprev, frag, dtype == 1, vs, mu, tag=i)
        assert ff < 0.02
    assert (W > 0).mean() > 0.03
    # fitness against the oracle's volume
    vol.upload(F, W)
    T_eval = _shift(S.compose_delta(poses[-1].astype(np.float64), [0.2, 0.9, 0.1], np.radians(3.0), [0.02, -0.01, 0.015]), 0 * o32)
    d = S.add_noise(S.raycast_depth(scene, T_eval.astype(np.float64), K, w, h), 777, sigma_rel=0.01, dropout=0.05)
    pts = np.ascontiguousarray(orc.backproject(d, K, 2).astype(np.float32))
    pst = S.sample_pst(500, 4321)
    scale = np.array([0.03, 0.05, 0.02, 0.04, 0.06, 0.03], dtype=np.float32)
    pose = _shift(poses[-1], o32)
    fit, cnt = vol.eval_particles(_dev(pts), _dev(pst), pose, scale)
    ref = orc.eval_particles(g, F, W, pts, pst, pose, scale, nthreads=8)
    assert 0 < ref["n"].max() and ref["n"].min() < ref["M_O"]
    _check_fitness(fit, cnt, ref, FIT_TOL[dtype])
    # read-out
    hit, frag_frac, _ = _raycast_compare(vol, g, F, W, K, w, h, pose, float(np.float32(0.04)), 5.0)
    assert hit > 0.2 and frag_frac < 0.05
    vol.destroy()


@pytest.mark.parametrize("dtype,w_max", [(0, 1), (0, 3), (1, 3)])
def test_weight_cap_and_running_average_beyond_it(dtype, w_max):
    """w_max < 255: weights saturate at the cap (min(W + 1, w_max)) and the value keeps averaging with factor
    w_max / (w_max + 1) -- the regime a long sequence reaches at 255.  Six frames of two alternating depths."""
    rf = _rf()
    dims, vs, mu = (48, 40, 56), 0.05, 0.15
    w, h = 96, 72
    K = np.array([80.0, 80.0, 47.5, 35.5], dtype=np.float32)
    g = orc.make_grid(dims, vs, mu)
    F, W = orc.empty_volume(dims)
    vol = rf.Volume(dims, vs, mu, dtype=dtype, w_max=w_max)
    ext = np.array(dims) * vs
    T = S.look_at(np.array([0.45, 0.5, -0.15]) * ext, np.array([0.5, 0.5, 0.8]) * ext).astype(np.float32)
    rng = np.random.Generator(np.random.Philox(9))
    for i in range(6):
        d = np.full((h, w), 1.6 + 0.07 * (i % 2), dtype=np.float32) + rng.normal(0, 0.004, (h, w)).astype(np.float32)
        Fprev, Wprev = F.copy(), W.copy()
        frag = np.zeros(F.size, dtype=np.uint8)
        orc.integrate(g, F, W, d, K, T, w_max=w_max, half_storage=(dtype == 1), nthreads=8, fragile=frag)
        vol.upload(Fprev, Wprev)
        vol.integrate(_dev(d), K, T)
        Ft, Wt = vol.download()
        # a voxel at the cap is updated although its weight does not move: compare it like an updated one
        check_integration(Ft, Wt, F, W, Wprev, frag, dtype == 1, vs, mu, tag=i)
        assert W.max() == min(i + 1, w_max)
    capped = (W == w_max) & (np.abs(F) < 0.999)
    assert capped.sum() > 1000                     # band voxels sit at the cap and kept moving
    vol.destroy()


def test_invalid_depth_values_are_skipped():
    """NaN, +inf, -inf, negative and zero depth are invalid pixels (A23): their voxels are not touched; a frame made only
    of such pixels changes nothing."""
    rf = _rf()
    dims, vs, mu = (70, 66, 50), 0.03, 0.09
    scene, K, w, h, poses, frames = _small_world(dims, vs, mu, n_frames=1)
    d = frames[0].copy()
    rng = np.random.Generator(np.random.Philox(5))
    kinds = rng.integers(0, 6, d.shape)
    d[kinds == 1] = np.nan
    d[kinds == 2] = np.inf
    d[kinds == 3] = -1.5
    d[kinds == 4] = -np.inf
    g = orc.make_grid(dims, vs, mu)
    F, W = orc.empty_volume(dims)
    Wprev = W.copy()
    frag = np.zeros(F.size, dtype=np.uint8)
    orc.integrate(g, F, W, d, K, poses[0], nthreads=8, fragile=frag)
    vol = rf.Volume(dims, vs, mu)
    vol.integrate(_dev(d), K, poses[0])
    Ft, Wt = vol.download()
    check_integration(Ft, Wt, F, W, Wprev, frag, False, vs, mu)
    assert 100 < (W > 0).sum() < 0.6 * (Wprev == 0).sum()
    # back-projection and the tracker's point sets skip them too
    pts = vol.backproject(_dev(d), K, 1).cpu().numpy()
    ref = orc.backproject(d, K, 1)
    assert np.array_equal(pts[:, 3], ref[:, 3]) and 0.2 < ref[:, 3].mean() < 0.5
    bad = np.full_like(d, np.nan)
    bad[::2] = -np.inf
    bad[::3] = 0.0
    before = vol.download()
    vol.integrate(_dev(bad), K, poses[0])
    after = vol.download()
    assert vol.last_updated() == 0 and all(np.array_equal(a, b) for a, b in zip(before, after))
    vol.destroy()


def test_f1_mode_inside_the_frame_loop_teacher_forced():
    """RF_TRACK_MODE_F1 (A6: rho = exp(-S / n), 0 when n < M_O / 2) through the same per-iteration gate as the default."""
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    vol = rf.Volume(dims, vs, mu, dtype=0)
    vol.upload(F, W)
    strides = (2, 4, 8)
    dp = [_dev(p) for p in psts]
    dd = _dev(depth)
    tol = FIT_TOL[0]
    ref = orc.pfo_track(g, F, W, depth, K, psts, strides, 6, T_prev, T_prev, r0=np.full(6, 0.06), early_stop=False, nthreads=8, mode=1)
    T32, r32 = T_prev.copy(), np.full(6, 0.06, dtype=np.float32)
    checked = 0
    for k in range(1, 7):
        l = (k - 1) % 3
        ev, up, M_O = _oracle_iteration(g, F, W, depth, K, psts[l], strides[l], T32, T_prev, r32, 0, mode=1)
        got = vol.pfo_track(dd, K, dp, strides, 1, T32, T_prev, r0=r32, flags=rf.RF_TRACK_NO_EARLY_STOP | rf.RF_TRACK_MODE_F1,
                            want_trace=True, start_iter=k - 1)
        gt = got["trace"][0]
        assert gt.M_O == M_O
        assert abs(gt.rho_ref - up.rho_ref) <= tol * up.rho_ref and abs(gt.rho_max - up.rho_max) <= tol * up.rho_max
        near = int(np.sum(np.abs(ev["rho"][1:] - up.rho_ref) <= 2 * tol * up.rho_ref))
        # F1 drops a candidate to 0 when fewer than half of its points can be sampled: one fragile point can flip that
        near += int(np.sum(np.abs(2 * ev["n"][1:].astype(np.int64) - M_O) <= 2 * ev["fragile"][1:]))
        assert abs(gt.n_aps - up.n_aps) <= near
        if up.n_aps - near > 0:
            bound = 4 * tol * up.rho_max * max(r32) * (up.n_aps + near) / up.sum_omega + 1e-7
            assert np.max(np.abs(np.array(gt.delta_star[:]) - np.array(up.delta_star[:]))) <= bound
            checked += 1
        row = ref["trace"][k - 1]
        T32 = np.array(row.pose[:], dtype=np.float32).reshape(3, 4)
        r32 = np.array(row.r[:], dtype=np.float32)
    assert checked >= 2
    # F1 and F2 are different fitness functions: the same start gives different reference fitness
    ref0 = orc.pfo_track(g, F, W, depth, K, psts, strides, 1, T_prev, T_prev, r0=np.full(6, 0.06), early_stop=False, nthreads=8)
    assert abs(ref0["trace"][0].rho_ref - ref["trace"][0].rho_ref) > 1e-3
    vol.destroy()


def test_two_empties_stop_rule_over_one_multi_iteration_call():
    """P:L306 inside ONE call: a swarm far too small to contain a better pose (r0 = 1e-5) finds an empty advantage set in
    iterations 1 and 2; the paper's rule re-inflates it after the first and stops after the second.  The CUDA loop and the
    oracle must agree on iters_run, stop, empty_run and the re-inflated axis lengths."""
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    vol = rf.Volume(dims, vs, mu, dtype=0)
    vol.upload(F, W)
    dp = [_dev(p) for p in psts]
    T0 = T_true.astype(np.float32)                     # start at the optimum: nothing in a 1e-5 swarm is better by rounding
    r0 = np.full(6, 1e-7, dtype=np.float32)
    got = vol.pfo_track(_dev(depth), K, dp, (2, 4, 8), 20, T0, T_prev, r0=r0, want_trace=True)
    ref = orc.pfo_track(g, F, W, depth, K, psts, (2, 4, 8), 20, T0, T_prev, r0=r0.astype(np.float64), nthreads=8)
    assert got["iters_run"] == ref["iters_run"]
    for a, b in zip(got["trace"], ref["trace"]):
        assert (a.stop, a.empty_run, a.level, a.M_O) == (b.stop, b.empty_run, b.level, b.M_O)
        if a.n_aps == 0 and b.n_aps == 0:
            assert np.allclose(a.r[:], b.r[:], rtol=0, atol=1e-5)
    last = got["trace"][-1]
    if last.stop == 1:
        assert last.empty_run == 2 and got["status"] & rf.RF_TRACK_STOP_EMPTY
    assert got["evals"] == ref["evals"] and got["final_count"] == ref["final_count"]
    vol.destroy()


def test_volume_create_defaults_and_argument_errors():
    rf = _rf()
    dims, vs, mu = (40, 40, 40), 0.05, 0.15
    scene, K, w, h, poses, frames = _small_world((70, 66, 50), 0.03, 0.09, n_frames=1)
    a = rf.Volume.create_default(dims, vs, mu)                    # rf_volume_create: fp32, origin 0, w_max 255, default stream
    b = rf.Volume(dims, vs, mu, dtype=rf.RF_F32_W8)
    for v in (a, b):
        v.integrate(_dev(frames[0]), K, poses[0])
    torch.cuda.synchronize()
    ta, wa = a.download()
    tb, wb = b.download()
    assert np.array_equal(ta, tb) and np.array_equal(wa, wb) and (wa > 0).sum() > 100
    # misaligned points: the fitness kernel stages point tiles with 16-byte bulk copies
    pst = _dev(S.sample_pst(16, 3))
    buf = torch.zeros(4 * 64 + 1, dtype=torch.float32, device="cuda")
    mis = buf[1:].view(64, 4)
    assert mis.data_ptr() % 16 == 4
    ident = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0]], dtype=np.float32)
    with pytest.raises(rf.RFError, match="aligned"):
        b.eval_particles(mis, pst, ident, np.ones(6, np.float32))
    with pytest.raises(rf.RFError):
        b.eval_particles(buf[:256].view(64, 4), pst, ident, np.ones(6, np.float32), mode=7)
    with pytest.raises(rf.RFError):
        rf.Volume(dims, vs, mu, w_max=300)
    with pytest.raises(rf.RFError):
        rf.Volume((9000, 8, 8), vs, mu)
    a.destroy(); b.destroy()


def test_stage_frame_slot_reuse_invalidates_the_consumed_frame():
    """rf_stage_frame re-uses the slot of the frame consumed two calls earlier: after that, rf_integrate_ex(depth_on_host = 2)
    must fail instead of fusing another frame's pixels."""
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    vol = rf.Volume(dims, vs, mu)
    vol.upload(F, W)
    dp = [_dev(p) for p in psts]
    pins = [torch.from_numpy(np.ascontiguousarray(depth + 0.01 * i)).pin_memory() for i in range(3)]
    r0 = np.full(6, 0.05, dtype=np.float32)
    vol.stage_frame(pins[0]); vol.stage_frame(pins[1])
    o = vol.pfo_track(tuple(depth.shape), K, dp, (2, 4, 8), 2, T_prev, T_prev, r0=r0)      # consumes frame 0
    vol.stage_frame(pins[2])                                                              # overwrites frame 0's slot
    with pytest.raises(rf.RFError):
        vol.integrate(None, K, o["pose"], staged_shape=depth.shape)
    vol.destroy()

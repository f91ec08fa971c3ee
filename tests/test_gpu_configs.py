"""GPU parity at BASELINE.json's full sizes (configs 2-5), in the launch configuration bench.py times.

The oracle cannot run the full problems in seconds, so each test compares what the oracle can compute one by one:
a seeded sample of particles over all points (particles are independent), a seeded sample of bricks over all frames
(voxels are independent), and the first iteration of a tracked frame (identical start state).  Volumes are built
by the ORACLE's integration (never by the CUDA path) and uploaded.
"""
import numpy as np
import pytest

import oracle as orc
import rf_synth as S
from gates import check_integration

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

NT = 16


def _rf():
    import paper_2105_05600_b200 as rf
    return rf


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _config3_world(first, count, mu, n_build):
    """Scene, true poses and noisy frames [first, first+count) of the config-3 sequence, and the 512^3 fp16 volume the
    oracle builds from the `n_build` frames before `first` at their true poses."""
    scene = S.make_config3_scene()
    traj = S.make_config3_trajectory(scene, n_frames=200)
    dims, vs = (512, 512, 512), 0.01
    g = orc.make_grid(dims, vs, mu)
    F, W = orc.empty_volume(dims)
    K = None
    for i in range(first - n_build, first):
        d, K = S.render_frame(scene, traj[i], 3, i)
        orc.integrate(g, F, W, d, K, traj[i].astype(np.float32), half_storage=True, nthreads=NT)
    frames = [S.render_frame(scene, traj[i], 3, i)[0] for i in range(first, first + count)]
    return dims, vs, g, F, W, K, traj, frames


def test_config4_fitness_cell_128k_x_64k_sampled():
    """Largest cell of the config-4 sweep: 131072 particles x 65536 points on a 512^3 fp16 volume, scale 0.1.
    Oracle parity on a seeded sample of 256 particles over ALL points; plus a small cell (1024 x 1024) in full."""
    rf = _rf()
    dims, vs, g, F, W, K, traj, frames = _config3_world(100, 1, 0.04, 6)
    vol = rf.Volume(dims, vs, 0.04, dtype=rf.RF_F16_W8)
    vol.upload(F, W)
    pts = orc.backproject(frames[0], K, 1).astype(np.float32)
    valid = np.flatnonzero(pts[:, 3] != 0)
    rng = np.random.Generator(np.random.Philox(S.config_seed(4, 8)))
    pst = S.sample_pst(131072, S.config_seed(4, 5))
    axis = rng.standard_normal(3)
    centre = S.compose_delta(traj[100], axis / np.linalg.norm(axis), np.radians(1.0), 0.02 * np.array([0.6, -0.64, 0.48])).astype(np.float32)
    scale = np.full(6, 0.1, dtype=np.float32)
    dpst = _dev(pst)
    for M, N in ((65536, 131072), (1024, 1024)):
        sel = np.sort(rng.choice(valid, size=M, replace=False))          # without replacement, scan order
        p = np.ascontiguousarray(pts[sel])
        fit, cnt = vol.eval_particles(_dev(p), dpst[:N], centre, scale)
        sample = np.sort(rng.choice(N, size=min(N, 256), replace=False))
        ref = orc.eval_particles(g, F, W, p, pst[sample], centre, scale, nthreads=NT)
        gf = fit.cpu().numpy().astype(np.float64)[sample]
        gn = cnt.cpu().numpy()[sample]
        assert ref["M_O"] == M
        assert np.all(np.abs(gn.astype(np.int64) - ref["n"]) <= ref["fragile"]), (M, N)
        rel = np.abs(gf - ref["rho"]) / np.maximum(ref["rho"], 1e-30)
        assert np.all(rel <= 2e-3 + 2.0 * ref["fragile"] / M), (M, N, rel.max())
        assert ref["n"].max() > 0.2 * M                                    # the sample is not vacuous
    vol.destroy()


def test_config5_integration_1024_cube_sampled_bricks():
    """1024^3 fp16+u8 volume, voxel 5 mm: 4 frames at seeded random poses, oracle parity on 4096 seeded 8^3 bricks
    (teacher-forced per frame on those bricks: the oracle's value before the frame is what the GPU had, bit for bit,
    whenever the previous frame matched)."""
    rf = _rf()
    dims, vs, mu = (1024, 1024, 1024), 0.005, 0.02
    scene = S.make_config3_scene()
    poses = S.make_config5_poses(scene, 4)
    g = orc.make_grid(dims, vs, mu)
    rng = np.random.Generator(np.random.Philox(S.config_seed(5, 8)))
    bricks = rng.choice(128 ** 3, size=4096, replace=False)
    bx, by, bz = bricks % 128, (bricks // 128) % 128, bricks // (128 * 128)
    l = np.arange(512)
    lx, ly, lz = l & 7, (l >> 3) & 7, l >> 6
    lin = ((bz[:, None] * 8 + lz) * 1024 + (by[:, None] * 8 + ly)) * 1024 + (bx[:, None] * 8 + lx)
    lin = np.sort(lin.reshape(-1).astype(np.int64))
    Fs = np.ones(lin.size, dtype=np.float32)
    Ws = np.zeros(lin.size, dtype=np.float32)
    ever = np.zeros(lin.size, dtype=np.uint8)             # voxels the oracle ever flagged fragile (R-I2): left out below
    vol = rf.Volume(dims, vs, mu, dtype=rf.RF_F16_W8)
    dlin = torch.from_numpy(lin).cuda()
    total_upd = 0
    dprev = np.zeros(lin.size)
    for i, T in enumerate(poses):
        d, K = S.render_frame(scene, T, 5, i)
        Wprev = Ws.copy()
        orc.integrate_subset(g, lin, Fs, Ws, d, K, T.astype(np.float32), half_storage=True, fragile=ever)
        vol.integrate(_dev(d), K, T.astype(np.float32))
        total_upd += vol.last_updated()
        t, w = vol.download_device()
        Ft, Wt = t[dlin].cpu().numpy(), w[dlin].cpu().numpy()
        del t, w
        # free-running over the frames (a 1024^3 volume is not re-uploaded per frame): every frame may add one rounding
        # step to what a voxel inherited (tests/gates.py)
        _, _, dprev = check_integration(Ft, Wt, Fs, Ws, Wprev, ever, True, vs, mu, tag=i, max_diff_frac=0.01 * (i + 1),
                                        d_prev=dprev, frames=i + 1)
    assert (Ws > 0).mean() > 0.01 and total_upd > 10_000_000 and ever.mean() < 0.02
    vol.destroy()


def test_config2_tracking_step_256_cube():
    """Config 2: 256^3 fp32 volume built by the oracle from 30 noisy frames, one 320x240 frame perturbed by 15 deg and
    8 cm, PST 1024/3072/10240, strides 4/8/16, exactly 20 iterations.  Iteration 1 (identical start state) must agree
    tightly; the free run must end where the oracle's ends (A20/A21)."""
    rf = _rf()
    c = S.make_config2_inputs()
    dims, vs, mu, K = c["dims"], c["voxel_size"], c["trunc"], c["K"]
    g = orc.make_grid(dims, vs, mu)
    F, W = orc.empty_volume(dims)
    for T, d in zip(c["build_poses"], c["build_frames"]):
        orc.integrate(g, F, W, d, K, T, nthreads=NT)
    vol = rf.Volume(dims, vs, mu, dtype=rf.RF_F32_W8)
    vol.upload(F, W)
    Tp = c["T_prev"]
    got = vol.pfo_track(_dev(c["tracked_depth"]), K, [_dev(p) for p in c["psts"]], c["strides"], 20, Tp, Tp, r0=None,
                        flags=rf.RF_TRACK_NO_EARLY_STOP, want_trace=True)
    ref = orc.pfo_track(g, F, W, c["tracked_depth"], K, c["psts"], c["strides"], 20, Tp, Tp, r0=None, early_stop=False,
                        nthreads=NT)
    assert got["iters_run"] == ref["iters_run"] == 20
    g1, o1 = got["trace"][0], ref["trace"][0]
    assert g1.M_O == o1.M_O and g1.level == 0
    assert abs(g1.rho_ref - o1.rho_ref) <= 1e-5 * o1.rho_ref
    assert abs(g1.rho_max - o1.rho_max) <= 1e-5 * o1.rho_max
    assert abs(g1.n_aps - o1.n_aps) <= max(2, o1.n_aps // 200)
    if o1.n_aps > 0:
        assert np.max(np.abs(np.array(g1.pose[:]) - np.array(o1.pose[:]))) <= 1e-4
    # evals = sum over iterations of (N_l + 1) * |O_k|, plus the centre-only evaluation of the first-frame rule (A11)
    assert sum(int(t.M_O) * (n + 1) for t, n in zip(got["trace"], [1024, 3072, 10240] * 7)) + g1.M_O == got["evals"]
    e_gpu = np.linalg.norm(got["pose"][:, 3] - c["T_true"][:, 3])
    e_orc = np.linalg.norm(ref["pose"][:, 3] - c["T_true"][:, 3])
    assert abs(e_gpu - e_orc) <= 0.02, (e_gpu, e_orc)
    assert abs(got["trace"][-1].rho_ref - ref["trace"][-1].rho_ref) <= 0.02
    vol.destroy()


def test_config3_sequence_teacher_forced_frames():
    """Config 3: 512^3 fp16+u8, 640x480 frames, strides 8/16/32, truncation 12 cm (DESIGN.md R-C3).  Three
    consecutive frames, teacher-forced per frame (A21): each frame both sides start from the oracle's pose and r0 and
    the oracle's volume; compared are iteration 1 (tightly), where the free run of the frame ends (loosely), and the
    frame's integration at the oracle's pose on 2048 seeded bricks."""
    rf = _rf()
    mu = 0.12
    dims, vs, g, F, W, K, traj, frames = _config3_world(30, 3, mu, 8)
    psts = [S.sample_pst(n, S.config_seed(3, 5 + i)) for i, n in enumerate((1024, 3072, 10240))]
    dp = [_dev(p) for p in psts]
    vol = rf.Volume(dims, vs, mu, dtype=rf.RF_F16_W8)
    vol.upload(F, W)
    rng = np.random.Generator(np.random.Philox(S.config_seed(3, 8)))
    bricks = rng.choice(64 ** 3, size=2048, replace=False)
    bx, by, bz = bricks % 64, (bricks // 64) % 64, bricks // (64 * 64)
    l = np.arange(512)
    lin = ((bz[:, None] * 8 + (l >> 6)) * 512 + (by[:, None] * 8 + ((l >> 3) & 7))) * 512 + (bx[:, None] * 8 + (l & 7))
    lin = np.sort(lin.reshape(-1).astype(np.int64))
    dlin = torch.from_numpy(lin).cuda()
    pose = traj[29].astype(np.float32)
    r0 = np.array([0.03, 0.03, 0.03, 0.15, 0.15, 0.15], dtype=np.float32)
    ever = np.zeros(F.size, dtype=np.uint8)                # union of the oracle's fragile flags over the frames so far
    dprev = np.zeros(lin.size)
    for i, d in enumerate(frames):
        got = vol.pfo_track(_dev(d), K, dp, (8, 16, 32), 20, pose, pose, r0=r0, want_trace=True)
        ref = orc.pfo_track(g, F, W, d, K, psts, (8, 16, 32), 20, pose, pose, r0=r0.astype(np.float64), nthreads=NT)
        g1, o1 = got["trace"][0], ref["trace"][0]
        assert g1.M_O == o1.M_O, i
        assert abs(g1.rho_ref - o1.rho_ref) <= 2e-3 * o1.rho_ref, i
        assert abs(g1.rho_max - o1.rho_max) <= 2e-3 * o1.rho_max, i
        te_g = np.linalg.norm(got["pose"][:, 3] - traj[30 + i][:, 3])
        te_o = np.linalg.norm(ref["pose"][:, 3] - traj[30 + i][:, 3])
        assert abs(te_g - te_o) <= 0.03, (i, te_g, te_o)
        # teacher: continue from the oracle's result
        pose, r0 = ref["pose"].astype(np.float32), ref["r1"].astype(np.float32)
        Fprev, Wprev = F[lin].copy(), W[lin].copy()
        orc.integrate(g, F, W, d, K, pose, half_storage=True, nthreads=NT, fragile=ever)
        vol.integrate(_dev(d), K, pose)
        t, w = vol.download_device()
        Ft, Wt = t[dlin].cpu().numpy(), w[dlin].cpu().numpy()
        del t, w
        # the volume is not re-uploaded between frames: every frame may add one rounding step to what a voxel inherited
        _, _, dprev = check_integration(Ft, Wt, F[lin], W[lin], Wprev, ever[lin], True, vs, mu, tag=i, max_diff_frac=0.01 * (i + 1),
                                        d_prev=dprev, frames=i + 1)
        assert (W[lin] != Wprev).sum() > 1000                            # the sampled bricks saw this frame
    vol.destroy()


def test_config3_raycast_readout_against_the_oracle_and_the_analytic_scene():
    """Read-out at config-3 size: 30 frames fused by rf_integrate at the true poses, then a 640x480 ray cast from the next
    pose: (1) parity with the oracle's ray cast of the downloaded volume, every pixel; (2) the read-out depth against the
    analytic scene's noise-free depth -- an end-to-end check of integration + read-out that involves neither side's
    arithmetic (frames carry 1 % depth noise, so the fused surface is within a voxel or so, not exact)."""
    rf = _rf()
    mu = 0.12
    scene = S.make_config3_scene()
    traj = S.make_config3_trajectory(scene, n_frames=200)
    dims, vs = (512, 512, 512), 0.01
    vol = rf.Volume(dims, vs, mu, dtype=rf.RF_F16_W8)
    K = None
    for i in range(30):
        d, K = S.render_frame(scene, traj[i], 3, i)
        vol.integrate(_dev(d), K, traj[i].astype(np.float32))
    pose = traj[30].astype(np.float32)
    step, z_max = float(np.float32(0.05)), 8.0
    d, n = vol.raycast(K, 640, 480, pose, step, z_max, want_normals=True)
    d, n = d.cpu().numpy(), n.cpu().numpy()
    F, W = vol.download()
    g = orc.make_grid(dims, vs, mu)
    od, on, frag = orc.raycast(g, F, W, K, 640, 480, pose, step, z_max, nthreads=NT)
    solid, hit = frag == 0, od > 0
    assert frag.mean() < 0.05 and hit.mean() > 0.5
    assert np.array_equal(d[solid] > 0, hit[solid])
    m = solid & hit
    assert np.max(np.abs(d[m] - od[m])) <= 1e-5
    fin = np.isfinite(on).all(-1) & m
    assert np.array_equal(np.isfinite(n).all(-1)[m], fin[m]) and np.max(np.abs(n[fin] - on[fin])) <= 1e-4
    clean = S.raycast_depth(scene, traj[30], K, 640, 480)
    both = (d > 0) & np.isfinite(clean) & (clean > 0)
    err = np.abs(d[both] - clean[both])
    assert both.mean() > 0.5
    assert np.median(err) < 0.5 * vs and np.quantile(err, 0.9) < 2.0 * vs, (np.median(err), np.quantile(err, 0.9))
    vol.destroy()

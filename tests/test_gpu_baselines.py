"""GPU parity of the Section 5.2 comparison methods (vanilla PFO, PSO) and of the A14 threshold variant.

The state updates are defined on binary32 state with fp64 arithmetic in a fixed order (reading B4), so proposal, PSO move
and bookkeeping are compared BIT FOR BIT; resampling is compared exactly on every slot that is not within the fitness
tolerance of a boundary of the cumulative weights; the fitness itself goes through the usual gate."""
import numpy as np
import pytest

import oracle as orc
import rf_synth as S
from gates import check_iteration
from test_gpu_parity import FIT_TOL, _check_fitness, _dev, _oracle_iteration, _rf, _track_world

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _vol(rf):
    return rf.Volume((16, 16, 16), 0.05, 0.15)


def test_propose_and_pso_move_are_bit_exact():
    rf = _rf()
    vol = _vol(rf)
    rng = np.random.Generator(np.random.Philox(314))
    N = 4099
    d = (rng.standard_normal((N, 6)) * np.array([0.4, 0.4, 0.4, 1.0, 1.0, 1.0])).astype(np.float32)      # many |q| > 0.95
    z = rng.standard_normal((N, 6)).astype(np.float32)
    sg = np.array([0.011, 0.02, 0.033, 0.1, 0.07, 0.05], dtype=np.float32)
    anc = np.sort(rng.integers(0, N, N)).astype(np.int32)
    for a in (None, anc):
        got = vol.baseline_propose(_dev(d), None if a is None else _dev(a), sg, _dev(z)).cpu().numpy()
        want = orc.baseline_propose(d, a, sg, z)
        assert np.array_equal(got, want) and (np.linalg.norm(want[:, :3], axis=1) <= 0.9500001).all()
        assert (np.linalg.norm(d[:, :3].astype(np.float64) + sg[:3] * z[:, :3], axis=1) > 0.95).sum() > 100      # the clamp was exercised
    x = (0.3 * rng.standard_normal((N, 6))).astype(np.float32)
    v = (0.05 * rng.standard_normal((N, 6))).astype(np.float32)
    pb = (0.3 * rng.standard_normal((N, 6))).astype(np.float32)
    gb = np.concatenate([0.2 * rng.standard_normal(6), [0.9, 17.0]]).astype(np.float32)
    ua, ub = rng.random((N, 6), dtype=np.float32), rng.random((N, 6), dtype=np.float32)
    xd, vd = _dev(x), _dev(v)
    vol.baseline_pso_move(xd, vd, _dev(pb), _dev(gb), _dev(ua), _dev(ub))
    xo, vo = orc.baseline_pso_move(x, v, pb, gb, ua, ub)
    assert np.array_equal(xd.cpu().numpy(), xo) and np.array_equal(vd.cpu().numpy(), vo)
    vol.destroy()


@pytest.mark.parametrize("N", [1, 37, 1024, 10240, 70001])
def test_systematic_resampling_matches_the_oracle(N):
    rf = _rf()
    vol = _vol(rf)
    rng = np.random.Generator(np.random.Philox(N))
    w = (rng.random(N) ** 6).astype(np.float32) + np.float32(1e-6)
    if N > 40:
        w[5:30] = 0.0                                    # zero-weight particles never get a slot
    for u in (0.0, 0.25, 0.9999):
        got = vol.baseline_resample(_dev(w), u).cpu().numpy()
        want, near = orc.systematic_resample(w.astype(np.float64), u, tol=1e-12)
        ok = near == 0
        assert np.array_equal(got[ok], want[ok]) and (~ok).sum() <= 2
        assert np.all(np.abs(got[~ok].astype(np.int64) - want[~ok]) <= 1)
        assert np.all(np.diff(got) >= 0) and (N <= 40 or not np.isin(got, np.arange(5, 30)).any())
    vol.destroy()


def test_best_bookkeeping_matches_the_oracle():
    rf = _rf()
    vol = _vol(rf)
    rng = np.random.Generator(np.random.Philox(99))
    N = 3001
    x = rng.standard_normal((N, 6)).astype(np.float32)
    pb_o, pf_o, g_o = np.zeros((N, 6), np.float32), np.zeros(N, np.float32), np.zeros(8, np.float32)
    pb_g, pf_g, g_g = _dev(pb_o), _dev(pf_o), _dev(g_o)
    for step in range(4):
        fit = np.round(rng.random(N), 2).astype(np.float32)          # two decimals: plenty of exact ties
        xs = (x + step).astype(np.float32)
        orc.baseline_best(fit, xs, pb_o, pf_o, step == 0, g_o)
        vol.baseline_best(_dev(fit), _dev(xs), pb_g, pf_g, step == 0, g_g)
        assert np.array_equal(pb_g.cpu().numpy(), pb_o) and np.array_equal(pf_g.cpu().numpy(), pf_o)
        assert np.array_equal(g_g.cpu().numpy(), g_o)
    g2_o, g2_g = np.zeros(8, np.float32), _dev(np.zeros(8, np.float32))      # without personal bests (vanilla PFO's run best)
    fit = np.round(rng.random(N), 1).astype(np.float32)
    orc.baseline_best(fit, x, None, None, True, g2_o)
    vol.baseline_best(_dev(fit), _dev(x), None, None, True, g2_g)
    assert np.array_equal(g2_g.cpu().numpy(), g2_o) and g2_o[7] == np.flatnonzero(fit == fit.max())[0]
    vol.destroy()


def test_vanilla_pfo_and_pso_steps_teacher_forced():
    """Five steps of each baseline on the 128^3 tracking world: every step both sides start from the oracle's state;
    fitness through the usual gate, resampling exact off the slots near a cumulative-weight boundary, state updates bit
    for bit.  Also: both methods improve the best fitness over the start pose (they are optimisers)."""
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    vol = rf.Volume(dims, vs, mu)
    vol.upload(F, W)
    tol = FIT_TOL[0]
    pts = orc.backproject(depth, K, 4).astype(np.float32)
    dpts = _dev(pts)
    ones = np.ones(6, dtype=np.float32)
    N = 1024
    rng = np.random.Generator(np.random.Philox(2718))
    sg = np.array([0.01, 0.01, 0.01, 0.01, 0.01, 0.01], dtype=np.float32)
    # ---- vanilla PFO
    state = np.zeros((N, 6), dtype=np.float32)
    anc = None
    best0 = None
    for k in range(5):
        z = rng.standard_normal((N, 6)).astype(np.float32)
        u = float(rng.random())
        prop_o = orc.baseline_propose(state, anc, sg, z)
        prop_g = vol.baseline_propose(_dev(state), None if anc is None else _dev(anc), sg, _dev(z))
        assert np.array_equal(prop_g.cpu().numpy(), prop_o)
        fit, cnt = vol.eval_particles(dpts, prop_g, T_prev, ones)
        ref = orc.eval_particles(g, F, W, pts, prop_o, T_prev, ones, nthreads=8)
        _check_fitness(fit, cnt, ref, tol)
        assert np.array_equal(ref["rho"], orc.eval_increments(g, F, W, pts, prop_o, T_prev, nthreads=8))
        anc_g = vol.baseline_resample(fit, u).cpu().numpy()
        anc_o, _ = orc.systematic_resample(ref["rho"], u)
        # a slot may legitimately take the neighbouring particle when it lies within the reach of the fitness tolerance of
        # a boundary of the cumulative weights: particle j's weight is known to tol_j = tol + 2 fragile_j / |O| (relative),
        # so boundary i moves by at most E_i = sum_{j<=i} w_j tol_j + C_i sum_j w_j tol_j
        wbar = ref["rho"] / ref["rho"].sum()
        e = np.cumsum(wbar * (tol + 2.0 * ref["fragile"] / max(ref["M_O"], 1)))
        C = np.cumsum(wbar)
        E = e + C * e[-1]
        um = (np.arange(N) + u) / N
        lo_c, lo_e = np.where(anc_o > 0, C[anc_o - 1], 0.0), np.where(anc_o > 0, E[anc_o - 1], 0.0)
        ok = (um - lo_c > lo_e) & ((C[anc_o] - um > E[anc_o]) | (anc_o == N - 1))
        assert np.array_equal(anc_g[ok], anc_o[ok]) and ok.mean() > 0.6
        assert np.all(np.abs(anc_g[~ok].astype(np.int64) - anc_o[~ok]) <= 2)
        best0 = ref["rho"].max() if best0 is None else best0
        state, anc = prop_o, anc_o
    assert ref["rho"].max() > best0 and ref["rho"].mean() > 0
    # ---- PSO from a small rescaled template
    x = (0.03 * psts[0][:N]).astype(np.float32)
    v = np.zeros((N, 6), dtype=np.float32)
    pb, pf, gb = np.zeros((N, 6), np.float32), np.zeros(N, np.float32), np.zeros(8, np.float32)
    gb_first = None
    for k in range(6):
        if k > 0:
            ua, ub = rng.random((N, 6), dtype=np.float32), rng.random((N, 6), dtype=np.float32)
            xd, vd = _dev(x), _dev(v)
            vol.baseline_pso_move(xd, vd, _dev(pb), _dev(gb), _dev(ua), _dev(ub))
            x, v = orc.baseline_pso_move(x, v, pb, gb, ua, ub)
            assert np.array_equal(xd.cpu().numpy(), x) and np.array_equal(vd.cpu().numpy(), v)
        fit, cnt = vol.eval_particles(dpts, _dev(x), T_prev, ones)
        ref = orc.eval_particles(g, F, W, pts, x, T_prev, ones, nthreads=8)
        _check_fitness(fit, cnt, ref, tol)
        # bookkeeping on the ORACLE's fitness (rounded to binary32) on both sides: the teacher state of the next step
        f32 = ref["rho"].astype(np.float32)
        pbd, pfd, gbd = _dev(pb), _dev(pf), _dev(gb)
        vol.baseline_best(_dev(f32), _dev(x), pbd, pfd, k == 0, gbd)
        orc.baseline_best(f32, x, pb, pf, k == 0, gb)
        assert np.array_equal(pbd.cpu().numpy(), pb) and np.array_equal(gbd.cpu().numpy(), gb)
        gb_first = gb[6] if gb_first is None else gb_first
    assert gb[6] > gb_first
    vol.destroy()


def test_threshold_variant_teacher_forced():
    """RF_TRACK_THRESH_EQ21 (A14 variant) through the per-iteration gate: the threshold of iteration k is the
    one the oracle carried out of iteration k-1 (Eq. 21's rho~, or the old threshold after an empty step)."""
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    vol = rf.Volume(dims, vs, mu, dtype=0)
    vol.upload(F, W)
    strides = (2, 4, 8)
    dp = [_dev(p) for p in psts]
    dd = _dev(depth)
    tol = FIT_TOL[0]
    T32, r32 = T_prev.copy(), np.full(6, 0.06, dtype=np.float32)
    thresh = float("nan")
    checked = carried = 0
    for k in range(1, 10):
        l = (k - 1) % 3
        ev, up0, M_O = _oracle_iteration(g, F, W, depth, K, psts[l], strides[l], T32, T_prev, r32, 0)
        t32 = float(np.float32(thresh)) if thresh == thresh else float("nan")
        up = orc.swarm_update(ev["rho"], psts[l], T32.astype(np.float64), r32.astype(np.float64), 0, variant=orc.VAR_THRESH_EQ21, thresh=t32)
        got = vol.pfo_track(dd, K, dp, strides, 1, T32, T_prev, r0=r32, flags=rf.RF_TRACK_NO_EARLY_STOP | rf.RF_TRACK_THRESH_EQ21,
                            want_trace=True, start_iter=k - 1, aps_threshold=0.0 if thresh != thresh else t32)
        gt = got["trace"][0]
        if thresh == thresh:
            assert gt.rho_ref == t32 == up.rho_ref                      # the carried value is used as it is
            carried += up.rho_ref != up0.rho_ref
        # same gate; rho_ref is exact here, so `near` counts the candidates within tol of the carried threshold
        checked += bool(check_iteration(gt, ev, up, M_O, tol, r32, T32, level=l, tag=k))
        want_next = up.rho_tilde if up.n_aps > 0 else up.rho_ref
        assert got["aps_threshold"] == pytest.approx(want_next, abs=8 * tol)
        thresh = want_next
        T32 = np.array(up.T_new[:], dtype=np.float32).reshape(3, 4)
        r32 = np.array(up.r_new[:], dtype=np.float32)
    assert checked >= 2 and carried >= 3
    # inside one multi-iteration call the device carries the threshold itself: trace row k uses row k-1's value
    multi = vol.pfo_track(dd, K, dp, strides, 6, T_prev, T_prev, r0=np.full(6, 0.06, dtype=np.float32),
                          flags=rf.RF_TRACK_NO_EARLY_STOP | rf.RF_TRACK_THRESH_EQ21, want_trace=True)
    for k in range(1, 6):
        prev = multi["trace"][k - 1]
        assert multi["trace"][k].rho_ref == (prev.rho_tilde if prev.n_aps > 0 else prev.rho_ref), k
    vol.destroy()

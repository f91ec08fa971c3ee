"""rf_gn_track_noalloc (the entry point that allocates nothing: its scratch is a static device array inside the library)
against the existing path rf_gn_track, on two calls in a row.

The two paths launch the same kernels with the same shapes and every fold is in a fixed order, so the results must be
bit-identical: the gate is equality (the tolerance of tests/test_gpu_gn.py, 1e-8, is the fallback named in the message).
The second call uses other points, another start and fewer iterations than the first, so that anything left in the shared
array by the first call (its pose, its stop flag, its longer trace, partial rows of more CTAs) would show.  The file is
named to be collected last: the suite runs with pytest -x."""
import numpy as np
import pytest

import oracle as orc
import rf_synth as S
from test_gpu_parity import _rf, _track_world

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _same(a, b, what):
    assert a["iters_run"] == b["iters_run"], what
    assert np.array_equal(a["pose"], b["pose"]), (what, np.max(np.abs(a["pose"] - b["pose"])), "tolerance of test_gpu_gn: 1e-8")
    for k, (x, y) in enumerate(zip(a["rows"], b["rows"])):
        assert x.n == y.n and x.cost == y.cost and x.step_norm == y.step_norm, (what, k)
        assert list(x.A) == list(y.A) and list(x.b) == list(y.b), (what, k)


def test_no_alloc_entry_point_matches_rf_gn_track_twice_in_a_row():
    rf = _rf()
    assert rf.gn_noalloc_scratch_bytes() == 256 + 64 * 360 + 592 * 32 * 8 == 174848
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    vol = rf.Volume(dims, vs, mu, dtype=rf.RF_F16_W8)
    vol.upload(F.astype(np.float16).astype(np.float32), W)
    pts_a = torch.from_numpy(orc.backproject(depth, K, 1).astype(np.float32)).cuda()        # 19200 points: 75 CTAs
    pts_b = torch.from_numpy(orc.backproject(depth, K, 4).astype(np.float32)).cuda()        # 1200 points: 5 CTAs
    T_a = S.compose_delta(T_true, [0.5, -0.3, 0.8], np.radians(2.0), [0.012, -0.01, 0.011])
    T_b = S.compose_delta(T_true, [-0.2, 0.7, 0.1], np.radians(1.0), [-0.008, 0.006, 0.01])
    # the existing path first (its scratch comes from cudaMalloc), then the static-scratch path twice in a row
    want_a = vol.gn_track(pts_a, T_a, 12)
    want_b = vol.gn_track(pts_b, T_b, 3)
    assert want_a["iters_run"] == 12 and want_a["rows"][0].n > 8000 and want_b["iters_run"] == 3
    assert want_a["rows"][-1].cost < 0.6 * want_a["rows"][0].cost                           # not vacuous: it minimised
    got_a = vol.gn_track_noalloc(pts_a, T_a, 12)
    got_b = vol.gn_track_noalloc(pts_b, T_b, 3)
    _same(got_a, want_a, "first call")
    _same(got_b, want_b, "second call (after a longer run on more points left its state in the shared array)")
    # a run that stops early (no valid point) leaves the stop flag set in the array: the next call must not see it
    stop = vol.gn_track_noalloc(torch.zeros((300, 4), device="cuda"), T_a, 5)
    assert stop["iters_run"] == 1 and stop["rows"][0].n == 0 and np.array_equal(stop["pose"], T_a)
    _same(vol.gn_track_noalloc(pts_a, T_a, 12), want_a, "after an early stop")
    # the limit: 64 iterations run, 65 are rejected with a message that names the limit
    full = vol.gn_track_noalloc(pts_b, T_b, 64)
    _same(full, vol.gn_track(pts_b, T_b, 64), "64 iterations")
    with pytest.raises(rf.RFError, match="RF_GN_NOALLOC_MAX_ITERS"):
        vol.gn_track_noalloc(pts_b, T_b, 65)
    # and a second volume (fp32) shares the same array
    vol32 = rf.Volume(dims, vs, mu, dtype=rf.RF_F32_W8)
    vol32.upload(F, W)
    _same(vol32.gn_track_noalloc(pts_a, T_a, 6), vol32.gn_track(pts_a, T_a, 6), "second volume")
    vol32.destroy()
    vol.destroy()

"""Several volumes driven from several host threads at once (the throughput mode of `bench.py --sequences`): the header
promises that the library keeps no mutable state outside an rf_volume (bar the atomic launch counter), so two sequences
tracked and fused concurrently, each on its own stream, must end with exactly the bits they end with when run alone."""
import threading

import numpy as np
import pytest

from test_gpu_parity import _dev, _rf, _track_world

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _sequence(rf, vol, depth_dev, K, psts_dev, T_prev, r0, reps):
    """reps x (track the frame from T_prev, fuse it at the tracked pose); returns every pose and the final volume."""
    poses = []
    for _ in range(reps):
        out = vol.track_integrate(depth_dev, K, psts_dev, (2, 4, 8), 9, T_prev, T_prev, r0=r0, flags=0)
        assert out["integrated"]
        poses.append(out["pose"].copy())
    F, W = vol.download()
    return poses, F, W


def test_two_volumes_on_two_threads_match_the_sequential_runs():
    rf = _rf()
    dims, vs, mu, g, F, W, K, depth, psts, T_prev, T_true = _track_world()
    r0s = [np.full(6, 0.06, dtype=np.float32), np.full(6, 0.04, dtype=np.float32)]     # two different searches
    reps = 6

    def fresh(stream):
        v = rf.Volume(dims, vs, mu, dtype=rf.RF_F16_W8, stream=stream)
        v.upload(F.astype(np.float16).astype(np.float32), W)
        return v

    # alone, one after the other
    want = []
    for r0 in r0s:
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            dd, dp = _dev(depth), [_dev(p) for p in psts]
            torch.cuda.synchronize()
            v = fresh(s)
            want.append(_sequence(rf, v, dd, K, dp, T_prev, r0, reps))
            v.destroy()
    # together
    l0 = rf.launch_count()
    streams = [torch.cuda.Stream() for _ in r0s]
    dd, dp = _dev(depth), [_dev(p) for p in psts]
    torch.cuda.synchronize()
    vols = [fresh(s) for s in streams]
    got, errs = [None] * len(r0s), []
    gate = threading.Barrier(len(r0s))

    def worker(i):
        try:
            gate.wait()
            got[i] = _sequence(rf, vols[i], dd, K, dp, T_prev, r0s[i], reps)
        except Exception as e:                                            # surfaced below: a thread's exception is otherwise lost
            errs.append(e)

    th = [threading.Thread(target=worker, args=(i,)) for i in range(len(r0s))]
    for t in th:
        t.start()
    for t in th:
        t.join()
    torch.cuda.synchronize()
    assert not errs, errs
    for (p_w, F_w, W_w), (p_g, F_g, W_g) in zip(want, got):
        assert all(np.array_equal(a, b) for a, b in zip(p_w, p_g))
        assert np.array_equal(W_w, W_g) and np.array_equal(F_w, F_g, equal_nan=True)
    assert not np.array_equal(want[0][0][-1], want[1][0][-1])            # the two sequences really are different work
    assert rf.launch_count() > l0
    for v in vols:
        v.destroy()

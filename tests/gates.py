"""Parity gates shared by the GPU tests.  No arithmetic of the method lives here."""
import numpy as np


def check_integration(Ft, Wt, F, W, Wprev, frag, half, vs, mu, tag="", max_diff_frac=0.01, d_prev=None, frames=1):
    """One frame fused by the CUDA path (Ft, Wt) against the oracle (F, W); Wprev = the oracle's weights before the frame.

    frag: the oracle's per-voxel fragile flags (R-I2): voxels whose pixel / z > 0 / band decision lies within the reach of
    a binary32 evaluation of the voxel's camera-frame position.
      weights  exact on every voxel that is not flagged; a flagged voxel is at most one update apart per frame;
      values   fp32 storage: |dF| <= 1e-4 * vs / mu (north_star: 1e-4 of voxel_size, normalised);
               fp16 storage: |dF| <= max(1 fp16 ulp of the oracle's value, that same bound), and bit-equal on all but
               max_diff_frac of the observed voxels (the oracle rounds the fp64 average to binary16, the kernel the
               binary32 one: they differ where the average sits within ~1e-6 relative of a rounding boundary);
      unobserved voxels read 1.0.
    Teacher-forced use (both sides start the frame from the same state): d_prev = None, frames = 1.
    Free-running use (the CUDA volume is not re-uploaded between frames): d_prev = the per-voxel |dF| this function
    returned for the previous frame, frames = number of frames so far, frag = union of the flags so far.  A voxel the frame
    updates may then carry W/(W+1) of its inherited difference (the running average damps it) plus this frame's one
    rounding step; a voxel the frame leaves alone keeps its difference; a flagged voxel may be `frames` updates apart.
    Returns (fragile fraction among the frame's candidate voxels, differing fraction, per-voxel |dF|)."""
    solid = frag == 0
    assert np.array_equal(Wt[solid], W[solid]), (tag, int((Wt[solid] != W[solid]).sum()))
    fr = ~solid
    if fr.any():
        assert np.all(np.abs(Wt[fr] - W[fr]) <= frames), tag
        if frames == 1:
            assert np.all(np.abs(Wt[fr] - Wprev[fr]) <= 1), tag
    seen = (W > 0) & solid
    tol = 1e-4 * vs / mu
    d = np.abs(Ft.astype(np.float64) - F.astype(np.float64))
    step = np.full(F.shape, tol)
    if half:
        step = np.maximum(np.spacing(np.abs(F).astype(np.float16)).astype(np.float64) * 1.0001, tol)
    if d_prev is None:
        bound = step
    else:
        upd = W != Wprev
        at_cap = (W == Wprev) & (Wprev > 0)          # a voxel at the weight cap may have been updated without W moving
        wp = Wprev.astype(np.float64)
        bound = np.where(upd | at_cap, d_prev * wp / (wp + 1.0) + step, d_prev)
        bound = np.maximum(bound, d_prev * (~upd))   # untouched voxels keep their difference exactly
    bad = seen & (d > bound)
    assert not bad.any(), (tag, int(bad.sum()), float((d[bad] / bound[bad]).max()))
    diff_frac = float((d[seen] > 0).mean()) if seen.any() else 0.0
    if half:
        assert diff_frac <= max_diff_frac, (tag, diff_frac)
    unseen = (W == 0) & solid
    assert np.all(Ft[unseen] == 1.0), tag
    touched = (W != Wprev) | fr
    frag_frac = float(fr.sum() / max(int(touched.sum()), 1))
    return frag_frac, diff_frac, d


def check_iteration(gt, ev, up, M_O, tol, r32, T32, level=None, tag=""):
    """One teacher-forced PFO iteration of the CUDA path (trace row gt) against the oracle's (ev = its candidate
    fitness values, up = its swarm update) from the same float32 state (A20, A21).  tol = the fitness tolerance.
      rho_ref, rho_max   relative tol;   |APS| within the number of candidates that sit within 2 tol of the threshold;
      delta*             A20: continuous in the fitness values -- an error tol*rho on every rho_j moves it by at most
                         4 tol rho_max N_aps max(r) / sum(omega);  rho~, r and the pose follow from that bound;
      empty APS          pose unchanged bit for bit, r within 4 tol, same empty_run / stop.
    Returns True when the non-empty branch was compared."""
    if level is not None:
        assert gt.level == level, tag
    assert gt.M_O == M_O, (tag, gt.M_O, M_O)
    assert abs(gt.rho_ref - up.rho_ref) <= tol * up.rho_ref, tag
    assert abs(gt.rho_max - up.rho_max) <= tol * up.rho_max, tag
    near = int(np.sum(np.abs(ev["rho"][1:] - up.rho_ref) <= 2 * tol * up.rho_ref))
    assert abs(gt.n_aps - up.n_aps) <= near, (tag, gt.n_aps, up.n_aps, near)
    rmax = float(np.max(r32))
    if up.n_aps - near > 0:
        ds_o, ds_g = np.array(up.delta_star[:]), np.array(gt.delta_star[:])
        bound = 4 * tol * up.rho_max * rmax * (up.n_aps + near) / up.sum_omega + 1e-7
        assert np.max(np.abs(ds_g - ds_o)) <= bound, (tag, np.max(np.abs(ds_g - ds_o)), bound)
        assert abs(gt.rho_tilde - up.rho_tilde) <= 4 * tol * up.rho_max * (up.n_aps + near) / up.sum_omega * (up.rho_max - up.rho_ref) + 2 * tol, tag
        nv = np.linalg.norm(ds_o)
        rb = 0.9 * ((1 - up.rho_tilde) * 2 * np.sqrt(6) * bound / max(nv, 1e-12) + abs(gt.rho_tilde - up.rho_tilde)) + 1e-7
        assert np.max(np.abs(np.array(gt.r[:]) - np.array(up.r_new[:]))) <= rb, (tag, rb)
        assert np.max(np.abs(np.array(gt.pose[:]) - np.array(up.T_new[:]))) <= 4 * bound * (1 + np.max(np.abs(T32))) + 1e-6, tag
        assert gt.empty_run == 0, tag
        return True
    if up.n_aps == 0 and gt.n_aps == 0:
        assert np.allclose(np.array(gt.pose[:]).reshape(3, 4), np.asarray(T32, dtype=np.float64), atol=0), tag
        assert np.allclose(gt.r[:], up.r_new[:], rtol=0, atol=4 * tol), tag
        assert gt.empty_run == up.empty_run and gt.stop == up.stop, tag
    return False

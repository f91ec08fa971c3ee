"""ctypes front-end of the CPU oracle (oracle/rf_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It imports nothing from the product package and shares no code with the CUDA path.
The shared object is compiled on first use with plain g++ (-O2, -ffp-contract=off: no fused
multiply-adds, so the fp64 arithmetic is the written one on every host).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "rf_oracle.cpp"
_LIB = _HERE / "liboracle.so"

TAU, EPS, BETA, STOP_TOL, EMPTY_STOP = 0, 1, 2, 3, 4
# ablation variants (rf_oracle.cpp ORC_VAR_*)
VAR_NO_OVERLAP, VAR_RESCALE_ISO, VAR_RESCALE_ANISO, VAR_THRESH_EQ21 = 1, 2, 4, 8


def build(force: bool = False) -> Path:
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".{os.getpid()}.tmp")
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", str(tmp), str(_SRC), "-lpthread"])
        os.replace(tmp, _LIB)
    return _LIB


class Grid(C.Structure):
    _fields_ = [("dims", C.c_int32 * 3), ("voxel_size", C.c_float), ("trunc", C.c_float),
                ("origin", C.c_float * 3)]


class UpdateOut(C.Structure):
    _fields_ = [("T_new", C.c_double * 12), ("r_new", C.c_double * 6), ("delta_star", C.c_double * 6),
                ("rho_ref", C.c_double), ("rho_max", C.c_double), ("rho_tilde", C.c_double),
                ("sum_omega", C.c_double), ("n_aps", C.c_int32), ("argmax", C.c_int32),
                ("empty_run", C.c_int32), ("stop", C.c_int32)]


class TraceRow(C.Structure):
    _fields_ = [("level", C.c_int32), ("M_O", C.c_int32), ("n_aps", C.c_int32), ("argmax", C.c_int32),
                ("stop", C.c_int32), ("empty_run", C.c_int32),
                ("rho_ref", C.c_double), ("rho_max", C.c_double), ("rho_tilde", C.c_double),
                ("sum_omega", C.c_double), ("delta_star", C.c_double * 6), ("pose", C.c_double * 12),
                ("r", C.c_double * 6)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        _lib.orc_const.restype = C.c_double
        _lib.orc_rho.restype = C.c_double
        _lib.orc_rho.argtypes = [C.c_double, C.c_int32, C.c_int32, C.c_int32]
        _lib.orc_round_to_half.restype = C.c_float
        _lib.orc_round_to_half.argtypes = [C.c_double]
        _lib.orc_lattice_count.restype = C.c_int32
        _lib.orc_backproject.restype = C.c_int32
        _lib.orc_trilinear.restype = C.c_int32
        _lib.orc_overlap_mask.restype = C.c_int32
        _lib.orc_pfo_track_v.restype = C.c_int32
        _lib.orc_pfo_track.restype = C.c_int32
        _lib.orc_integrate_eps_p.restype = C.c_double
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def make_grid(dims, voxel_size, trunc, origin=(0.0, 0.0, 0.0)) -> Grid:
    g = Grid()
    g.dims[:] = [int(d) for d in dims]
    g.voxel_size = float(voxel_size)
    g.trunc = float(trunc)
    g.origin[:] = [float(o) for o in origin]
    return g


def const(which: int) -> float:
    return float(lib().orc_const(C.c_int(which)))


def rho(S: float, n: int, M_O: int, mode: int = 0) -> float:
    return float(lib().orc_rho(float(S), int(n), int(M_O), int(mode)))


def round_to_half(v: float) -> float:
    return float(lib().orc_round_to_half(float(v)))


def quat_to_R(q) -> np.ndarray:
    q = _f64(q)
    R = np.zeros(9)
    lib().orc_quat_to_R(_p(q, C.c_double), _p(R, C.c_double))
    return R.reshape(3, 3)


def apply_delta(T, delta) -> np.ndarray:
    T = _f64(T).reshape(12)
    d = _f64(delta)
    out = np.zeros(12)
    lib().orc_apply_delta(_p(T, C.c_double), _p(d, C.c_double), _p(out, C.c_double))
    return out.reshape(3, 4)


def pose_from_particle(T_c, r, p) -> np.ndarray:
    T = _f64(T_c).reshape(12)
    r = _f64(r)
    p = _f32(p)
    out = np.zeros(12)
    lib().orc_pose_from_particle(_p(T, C.c_double), _p(r, C.c_double), _p(p, C.c_float), _p(out, C.c_double))
    return out.reshape(3, 4)


def lattice_count(n: int, s: int) -> int:
    return int(lib().orc_lattice_count(C.c_int32(n), C.c_int32(s)))


def backproject(depth, K, stride: int) -> np.ndarray:
    """-> float64 [M,4] (x, y, z, mask)."""
    depth = _f32(depth)
    h, w = depth.shape
    K = _f32(K)
    m = lattice_count(w, stride) * lattice_count(h, stride)
    pts = np.zeros((max(m, 1), 4))
    got = lib().orc_backproject(_p(depth, C.c_float), C.c_int32(w), C.c_int32(h), _p(K, C.c_float),
                                C.c_int32(stride), _p(pts, C.c_double))
    assert got == m
    return pts[:m]


def trilinear(grid: Grid, tsdf, weight, xw):
    """-> (valid, psi, fragile)"""
    tsdf, weight, xw = _f32(tsdf), _f32(weight), _f64(xw)
    psi = C.c_double(0.0)
    frag = C.c_int32(0)
    ok = lib().orc_trilinear(C.byref(grid), _p(tsdf, C.c_float), _p(weight, C.c_float), _p(xw, C.c_double),
                             C.byref(psi), C.byref(frag))
    return bool(ok), psi.value, int(frag.value)


def eval_particles(grid: Grid, tsdf, weight, points, pst, pose, scale, mode: int = 0, nthreads: int = 1):
    """rf_eval_particles equivalent -> dict(S, n, fragile, rho, M_O)."""
    tsdf, weight = _f32(tsdf), _f32(weight)
    points, pst = _f32(points).reshape(-1, 4), _f32(pst).reshape(-1, 6)
    pose, scale = _f32(pose).reshape(12), _f32(scale).reshape(6)
    M, N = points.shape[0], pst.shape[0]
    S = np.zeros(N)
    n = np.zeros(N, dtype=np.int32)
    fr = np.zeros(N, dtype=np.int32)
    rh = np.zeros(N)
    M_O = C.c_int32(0)
    lib().orc_eval_particles(C.byref(grid), _p(tsdf, C.c_float), _p(weight, C.c_float), _p(points, C.c_float),
                             C.c_int32(M), _p(pst, C.c_float), C.c_int32(N), _p(pose, C.c_float),
                             _p(scale, C.c_float), C.c_int32(mode), C.c_int32(nthreads), _p(S, C.c_double),
                             _p(n, C.c_int32), _p(fr, C.c_int32), _p(rh, C.c_double), C.byref(M_O))
    return dict(S=S, n=n, fragile=fr, rho=rh, M_O=int(M_O.value))


def overlap_mask(pts, T_km1, T_prev, K, w: int, h: int):
    pts = _f64(pts).reshape(-1, 4)
    T1, T0 = _f64(T_km1).reshape(12), _f64(T_prev).reshape(12)
    K = _f32(K)
    keep = np.zeros(pts.shape[0], dtype=np.uint8)
    cnt = lib().orc_overlap_mask(_p(pts, C.c_double), C.c_int32(pts.shape[0]), _p(T1, C.c_double),
                                 _p(T0, C.c_double), _p(K, C.c_float), C.c_int32(w), C.c_int32(h),
                                 _p(keep, C.c_uint8))
    return keep, int(cnt)


def swarm_update(rho_all, pst, T, r, empty_run: int = 0, variant: int = 0, thresh: float = float("nan")) -> UpdateOut:
    """thresh: with VAR_THRESH_EQ21, the advantage-set threshold carried from the previous iteration (NaN = rho_all[0])."""
    rho_all = _f64(rho_all)
    pst = _f32(pst).reshape(-1, 6)
    assert rho_all.shape[0] == pst.shape[0] + 1
    T, r = _f64(T).reshape(12), _f64(r)
    out = UpdateOut()
    lib().orc_swarm_update_t(_p(rho_all, C.c_double), _p(pst, C.c_float), C.c_int32(pst.shape[0]),
                             _p(T, C.c_double), _p(r, C.c_double), C.c_int32(empty_run), C.c_int32(variant),
                             C.c_double(thresh), C.byref(out))
    return out


def pfo_track(grid: Grid, tsdf, weight, depth, K, psts, strides, iters: int, pose, prev_pose, r0=None,
              early_stop: bool = True, mode: int = 0, nthreads: int = 1, variant: int = 0):
    """Algorithm 1 for one frame -> dict(pose, r1, iters_run, trace (list of TraceRow), final_rho,
    final_count, evals)."""
    tsdf, weight, depth, K = _f32(tsdf), _f32(weight), _f32(depth), _f32(K)
    h, w = depth.shape
    psts = [_f32(p).reshape(-1, 6) for p in psts]
    pp = (C.POINTER(C.c_float) * 3)(*[_p(p, C.c_float) for p in psts])
    N = (C.c_int32 * 3)(*[p.shape[0] for p in psts])
    st = (C.c_int32 * 3)(*[int(s) for s in strides])
    pose_io = _f64(pose).reshape(12).copy()
    prev = _f64(prev_pose).reshape(12)
    has_r0 = C.c_int32(0 if r0 is None else 1)
    r0_io = np.zeros(6) if r0 is None else _f64(r0).copy()
    trace = (TraceRow * iters)()
    frho, fcnt, evals = C.c_double(0), C.c_int32(0), C.c_int64(0)
    k = lib().orc_pfo_track_v(C.byref(grid), _p(tsdf, C.c_float), _p(weight, C.c_float), _p(depth, C.c_float),
                              C.c_int32(w), C.c_int32(h), _p(K, C.c_float), pp, N, st, C.c_int32(iters),
                              C.c_int32(1 if early_stop else 0), C.c_int32(mode), C.c_int32(variant), C.c_int32(nthreads),
                              _p(pose_io, C.c_double), _p(prev, C.c_double), _p(r0_io, C.c_double),
                              C.byref(has_r0), trace, C.byref(frho), C.byref(fcnt), C.byref(evals))
    return dict(pose=pose_io.reshape(3, 4), r1=r0_io, iters_run=int(k), trace=[trace[i] for i in range(k)],
                final_rho=frho.value, final_count=int(fcnt.value), evals=int(evals.value))


def _fragile_arg(fragile, n):
    if fragile is None:
        return None
    assert fragile.dtype == np.uint8 and fragile.flags.c_contiguous and fragile.size == n
    return _p(fragile, C.c_uint8)


def integrate(grid: Grid, tsdf, weight, depth, K, pose, w_max: int = 255, half_storage: bool = False,
              nthreads: int = 1, fragile=None):
    """In-place update of float32 arrays tsdf / weight (dense, x-fastest).  fragile: optional uint8 array of the same
    size; voxels whose decisions a binary32 evaluation could take the other way (R-I2) are SET to 1 (never cleared)."""
    assert tsdf.dtype == np.float32 and weight.dtype == np.float32
    assert tsdf.flags.c_contiguous and weight.flags.c_contiguous
    depth, K, pose = _f32(depth), _f32(K), _f32(pose).reshape(12)
    h, w = depth.shape
    lib().orc_integrate(C.byref(grid), _p(tsdf, C.c_float), _p(weight, C.c_float), _p(depth, C.c_float),
                        C.c_int32(w), C.c_int32(h), _p(K, C.c_float), _p(pose, C.c_float), C.c_int32(w_max),
                        C.c_int32(1 if half_storage else 0), C.c_int32(nthreads), _fragile_arg(fragile, tsdf.size))


def integrate_subset(grid: Grid, lin_idx, tsdf_sub, weight_sub, depth, K, pose, w_max: int = 255,
                     half_storage: bool = False, fragile=None):
    lin = np.ascontiguousarray(lin_idx, dtype=np.int64)
    assert tsdf_sub.dtype == np.float32 and weight_sub.dtype == np.float32
    depth, K, pose = _f32(depth), _f32(K), _f32(pose).reshape(12)
    h, w = depth.shape
    lib().orc_integrate_subset(C.byref(grid), _p(lin, C.c_int64), C.c_int64(lin.shape[0]), _p(tsdf_sub, C.c_float),
                               _p(weight_sub, C.c_float), _p(depth, C.c_float), C.c_int32(w), C.c_int32(h),
                               _p(K, C.c_float), _p(pose, C.c_float), C.c_int32(w_max),
                               C.c_int32(1 if half_storage else 0), _fragile_arg(fragile, tsdf_sub.size))


def raycast(grid: Grid, tsdf, weight, K, w: int, h: int, pose, step: float, z_max: float, want_normals: bool = True,
            nthreads: int = 1):
    """-> (depth [h,w] f64, normals [h,w,3] f64 or None, fragile [h,w] u8)   (O9)"""
    tsdf, weight, K, pose = _f32(tsdf), _f32(weight), _f32(K), _f32(pose).reshape(12)
    depth = np.zeros((h, w), dtype=np.float64)
    normals = np.zeros((h, w, 3), dtype=np.float64) if want_normals else None
    frag = np.zeros((h, w), dtype=np.uint8)
    lib().orc_raycast(C.byref(grid), _p(tsdf, C.c_float), _p(weight, C.c_float), _p(K, C.c_float), C.c_int32(w),
                      C.c_int32(h), _p(pose, C.c_float), C.c_double(step), C.c_double(z_max), _p(depth, C.c_double),
                      _p(normals, C.c_double) if want_normals else None, _p(frag, C.c_uint8), C.c_int32(nthreads))
    return depth, normals, frag


# ---- baselines of Section 5.2 (vanilla PFO, PSO); every random number is an input
def baseline_propose(delta_in, ancestors, sigma, normals) -> np.ndarray:
    """Eq. (12) + clamp: float32 [N,6] -> float32 [N,6]."""
    d, z, sg = _f32(delta_in).reshape(-1, 6), _f32(normals).reshape(-1, 6), _f32(sigma).reshape(6)
    N = d.shape[0]
    anc = None if ancestors is None else np.ascontiguousarray(ancestors, dtype=np.int32)
    out = np.zeros((N, 6), dtype=np.float32)
    lib().orc_baseline_propose(_p(d, C.c_float), None if anc is None else _p(anc, C.c_int32), _p(sg, C.c_float),
                               _p(z, C.c_float), C.c_int32(N), _p(out, C.c_float))
    return out


def systematic_resample(weights, u: float, tol: float = 0.0):
    """-> (ancestors int32 [N], near uint8 [N])"""
    w = _f64(weights)
    N = w.shape[0]
    anc = np.zeros(N, dtype=np.int32)
    near = np.zeros(N, dtype=np.uint8)
    lib().orc_systematic_resample(_p(w, C.c_double), C.c_int32(N), C.c_double(u), C.c_double(tol), _p(anc, C.c_int32),
                                  _p(near, C.c_uint8))
    return anc, near


def pso_const(which: int) -> float:
    lib().orc_pso_const.restype = C.c_double
    return float(lib().orc_pso_const(C.c_int(which)))


def baseline_pso_move(x, v, pbest, gbest, ua, ub):
    """In place on float32 copies; returns (x, v)."""
    x, v = _f32(x).reshape(-1, 6).copy(), _f32(v).reshape(-1, 6).copy()
    pb, gb = _f32(pbest).reshape(-1, 6), _f32(gbest).reshape(-1)[:6].copy()
    a, b = _f32(ua).reshape(-1, 6), _f32(ub).reshape(-1, 6)
    lib().orc_baseline_pso_move(_p(x, C.c_float), _p(v, C.c_float), _p(pb, C.c_float), _p(gb, C.c_float), _p(a, C.c_float),
                                _p(b, C.c_float), C.c_int32(x.shape[0]))
    return x, v


def baseline_best(fitness, x, pbest, pbest_fit, first: bool, gbest):
    """In place on the float32 arrays pbest / pbest_fit (or None) and gbest [8]."""
    f, x = _f32(fitness), _f32(x).reshape(-1, 6)
    for a in (pbest, pbest_fit, gbest):
        assert a is None or (a.dtype == np.float32 and a.flags.c_contiguous)
    lib().orc_baseline_best(_p(f, C.c_float), _p(x, C.c_float), C.c_int32(f.shape[0]), None if pbest is None else _p(pbest, C.c_float),
                            None if pbest_fit is None else _p(pbest_fit, C.c_float), C.c_int32(1 if first else 0), _p(gbest, C.c_float))


def eval_increments(grid: Grid, tsdf, weight, points, delta, pose, mode: int = 0, nthreads: int = 1) -> np.ndarray:
    """Fitness of explicit float32 increments about `pose` (scale 1, every valid point) -> float64 [N]."""
    tsdf, weight = _f32(tsdf), _f32(weight)
    points, delta, pose = _f32(points).reshape(-1, 4), _f32(delta).reshape(-1, 6), _f32(pose).reshape(12)
    rho = np.zeros(delta.shape[0])
    lib().orc_eval_increments(C.byref(grid), _p(tsdf, C.c_float), _p(weight, C.c_float), _p(points, C.c_float),
                              C.c_int32(points.shape[0]), _p(delta, C.c_float), C.c_int32(delta.shape[0]), _p(pose, C.c_float),
                              C.c_int32(mode), C.c_int32(nthreads), _p(rho, C.c_double))
    return rho


def surface_points(grid: Grid, tsdf, weight, cap: int = 1 << 24):
    """O10: zero crossings along grid edges (the vertex set of marching cubes) -> (points float64 [n,3], edge keys int64 [n])."""
    tsdf, weight = _f32(tsdf), _f32(weight)
    pts = np.zeros((cap, 3), dtype=np.float64)
    edge = np.zeros(cap, dtype=np.int64)
    lib().orc_surface_points.restype = C.c_int64
    n = int(lib().orc_surface_points(C.byref(grid), _p(tsdf, C.c_float), _p(weight, C.c_float), _p(pts, C.c_double),
                                     _p(edge, C.c_int64), C.c_int64(cap)))
    assert n <= cap, "surface_points: capacity too small"
    return pts[:n].copy(), edge[:n].copy()


class GNRow(C.Structure):
    _fields_ = [("cost", C.c_double), ("n", C.c_int32), ("pad", C.c_int32), ("step_norm", C.c_double),
                ("A", C.c_double * 36), ("b", C.c_double * 6)]


def trilinear_grad(grid: Grid, tsdf, weight, xw):
    """-> (valid, psi, grad[3] per metre): the trilinear interpolant and its analytic derivative (O11)."""
    tsdf, weight, xw = _f32(tsdf), _f32(weight), _f64(xw)
    psi = C.c_double(0.0)
    gr = np.zeros(3)
    ok = lib().orc_trilinear_grad(C.byref(grid), _p(tsdf, C.c_float), _p(weight, C.c_float), _p(xw, C.c_double), C.byref(psi),
                                  _p(gr, C.c_double))
    return bool(ok), psi.value, gr


def gn_track(grid: Grid, tsdf, weight, points, pose, iters: int):
    """O11: Gauss-Newton on Eq. (4) -> dict(pose [3,4] f64, iters_run, rows (list of GNRow))."""
    tsdf, weight, points = _f32(tsdf), _f32(weight), _f32(points).reshape(-1, 4)
    pose_io = _f64(pose).reshape(12).copy()
    rows = (GNRow * iters)()
    k = lib().orc_gn_track(C.byref(grid), _p(tsdf, C.c_float), _p(weight, C.c_float), _p(points, C.c_float),
                           C.c_int32(points.shape[0]), _p(pose_io, C.c_double), C.c_int32(iters), rows)
    return dict(pose=pose_io.reshape(3, 4), iters_run=int(k), rows=[rows[i] for i in range(int(k))])


def integrate_eps_p() -> float:
    """Reach (metres) of a binary32 evaluation of a camera-frame voxel position, the fragile-voxel tolerance (R-I2)."""
    return float(lib().orc_integrate_eps_p())


def empty_volume(dims):
    n = int(dims[0]) * int(dims[1]) * int(dims[2])
    return np.ones(n, dtype=np.float32), np.zeros(n, dtype=np.float32)

"""Thin Python binding of include/rosefusion_b200.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of librosefusion_b200.so; PyTorch supplies device
memory and the stream.  There is no CPU fallback: if the library cannot be loaded this module raises.
Function names follow the C ABI (rf_volume_create -> Volume(...), rf_integrate -> Volume.integrate, ...).
"""
from __future__ import annotations

import ctypes as C
from typing import Optional, Sequence

import numpy as np
import torch

from . import build as _build

RF_F32_W8, RF_F16_W8 = 0, 1
RF_TRACK_NO_EARLY_STOP, RF_TRACK_MODE_F1, RF_TRACK_NO_GRAPH, RF_TRACK_NO_PDL = 1, 2, 4, 8
RF_TRACK_NO_OVERLAP, RF_TRACK_RESCALE_ISO, RF_TRACK_RESCALE_ANISO, RF_TRACK_MODE_EQ14, RF_TRACK_THRESH_EQ21 = 16, 32, 64, 128, 256
RF_TRACK_NO_POINTS, RF_TRACK_STOP_EMPTY, RF_TRACK_STOP_SMALL = 1, 2, 4

EXPORTS = [
    "rf_volume_create", "rf_volume_create_ex", "rf_volume_destroy", "rf_volume_reset", "rf_integrate",
    "rf_integrate_ex", "rf_stage_frame", "rf_integrate_last_updated", "rf_integrate_last_stats", "rf_backproject", "rf_eval_particles",
    "rf_eval_particles_ex", "rf_pfo_track", "rf_track_integrate", "rf_shard_begin", "rf_shard_eval", "rf_shard_apply", "rf_shard_end", "rf_volume_download", "rf_volume_download_ex",
    "rf_volume_upload", "rf_volume_download_box", "rf_volume_pool_stats", "rf_raycast", "rf_extract_surface_points", "rf_gn_track", "rf_gn_track_noalloc", "rf_gn_noalloc_scratch_bytes", "rf_baseline_propose", "rf_baseline_resample", "rf_baseline_pso_move", "rf_baseline_best", "rf_microbench_l2", "rf_profile_enable", "rf_profile_read", "rf_profile_read_launches", "rf_launch_count",
    "rf_last_error", "rf_version",
]


class RFError(RuntimeError):
    pass


class GNRow(C.Structure):
    """rf_gn_row."""
    _fields_ = [("cost", C.c_double), ("n", C.c_int32), ("pad", C.c_int32), ("step_norm", C.c_double),
                ("A", C.c_double * 36), ("b", C.c_double * 6)]


class VolumeOpts(C.Structure):
    _fields_ = [("dtype", C.c_int32), ("origin", C.c_float * 3), ("w_max", C.c_int32), ("stream", C.c_void_p),
                ("pool_bricks", C.c_int32)]


class Frame(C.Structure):
    _fields_ = [("depth", C.c_void_p), ("depth_on_host", C.c_int32), ("width", C.c_int32), ("height", C.c_int32),
                ("K", C.c_float * 4)]


class PstSet(C.Structure):
    _fields_ = [("pst_dev", C.c_void_p * 3), ("N", C.c_int32 * 3), ("stride", C.c_int32 * 3)]


class TrackState(C.Structure):
    _fields_ = [("pose_c2w", C.c_float * 12), ("prev_pose_c2w", C.c_float * 12), ("r0", C.c_float * 6),
                ("has_r0", C.c_int32), ("flags", C.c_int32), ("start_iter", C.c_int32), ("aps_threshold", C.c_float)]


class TrackResult(C.Structure):
    _fields_ = [("iters_run", C.c_int32), ("status", C.c_int32), ("final_fitness", C.c_float),
                ("final_count", C.c_int32), ("argmax", C.c_int32), ("evals", C.c_int64)]


class TrackTrace(C.Structure):
    _fields_ = [("level", C.c_int32), ("M_O", C.c_int32), ("n_aps", C.c_int32), ("argmax", C.c_int32),
                ("stop", C.c_int32), ("empty_run", C.c_int32),
                ("rho_ref", C.c_double), ("rho_max", C.c_double), ("rho_tilde", C.c_double),
                ("sum_omega", C.c_double), ("delta_star", C.c_double * 6), ("pose", C.c_double * 12),
                ("r", C.c_double * 6)]


_lib = None


def lib():
    """Load (building in-tree if stale) the C-ABI library.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        path = _build.build()
        try:
            _lib = C.CDLL(str(path))
        except OSError as e:      # loud failure: no fallback path exists
            raise RFError(f"cannot load {path}: {e}") from e
        _lib.rf_last_error.restype = C.c_char_p
        _lib.rf_launch_count.restype = C.c_int64
        _lib.rf_gn_noalloc_scratch_bytes.restype = C.c_int64
        for name in EXPORTS:
            getattr(_lib, name)
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise RFError(f"{what} failed (status {rc}): {lib().rf_last_error().decode()}")


def _f32p(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _host_f32(a, n: int) -> np.ndarray:
    out = np.ascontiguousarray(np.asarray(a, dtype=np.float32).reshape(-1))
    assert out.size == n
    return out


def _dev(t: torch.Tensor, dtype) -> int:
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise RFError("expected a contiguous CUDA tensor of dtype %s" % dtype)
    return t.data_ptr()


class Volume:
    """rf_volume: a bricked TSDF + weight volume resident in HBM."""

    def __init__(self, dims: Sequence[int], voxel_size: float, trunc: float, dtype: int = RF_F32_W8,
                 origin=(0.0, 0.0, 0.0), w_max: int = 255, stream: Optional[torch.cuda.Stream] = None, pool_bricks: int = 0):
        """pool_bricks > 0: a sparse volume (rf_volume_opts.pool_bricks) -- `dims` is a logical index space and at most that
        many 8x8x8 bricks are stored, allocated when an integration first sweeps them."""
        if not torch.cuda.is_available():
            raise RFError("no CUDA device: the ROSEFusion path has no CPU fallback")
        self.dims = tuple(int(d) for d in dims)
        self.voxel_size, self.trunc, self.dtype = float(voxel_size), float(trunc), int(dtype)
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        opts = VolumeOpts()
        opts.dtype = dtype
        opts.origin[:] = [float(o) for o in origin]
        opts.w_max = int(w_max)
        opts.stream = self.stream.cuda_stream
        opts.pool_bricks = int(pool_bricks)
        self.pool_bricks = int(pool_bricks)
        self._h = C.c_void_p()
        d = (C.c_int32 * 3)(*self.dims)
        _check(lib().rf_volume_create_ex(d, C.c_float(voxel_size), C.c_float(trunc), C.byref(opts), C.byref(self._h)),
               "rf_volume_create")

    @classmethod
    def create_default(cls, dims: Sequence[int], voxel_size: float, trunc: float) -> "Volume":
        """rf_volume_create: the five-argument call of north_star (fp32 TSDF, origin 0, w_max 255, legacy default stream)."""
        if not torch.cuda.is_available():
            raise RFError("no CUDA device: the ROSEFusion path has no CPU fallback")
        self = cls.__new__(cls)
        self.dims = tuple(int(d) for d in dims)
        self.voxel_size, self.trunc, self.dtype = float(voxel_size), float(trunc), RF_F32_W8
        self.stream = torch.cuda.default_stream()
        self._h = C.c_void_p()
        d = (C.c_int32 * 3)(*self.dims)
        _check(lib().rf_volume_create(d, C.c_float(voxel_size), C.c_float(trunc), C.byref(self._h)), "rf_volume_create")
        return self

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().rf_volume_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def reset(self):
        _check(lib().rf_volume_reset(self._h), "rf_volume_reset")

    # ---- a6
    def integrate(self, depth, K, pose_c2w, staged_shape=None):
        """depth: CUDA float32 tensor (H,W), or a host numpy / CPU tensor (then the H2D copy is part of the call), or
        None with staged_shape=(H,W): fuse the frame the last host-depth call already copied to the device."""
        K = _host_f32(K, 4)
        pose = _host_f32(pose_c2w, 12)
        if depth is None:
            h, w = staged_shape
            _check(lib().rf_integrate_ex(self._h, C.c_void_p(0), C.c_int32(2), C.c_int32(w), C.c_int32(h), _f32p(K), _f32p(pose)),
                   "rf_integrate_ex")
        elif isinstance(depth, torch.Tensor) and depth.is_cuda:
            h, w = depth.shape
            _check(lib().rf_integrate(self._h, C.c_void_p(_dev(depth, torch.float32)), C.c_int32(w), C.c_int32(h),
                                      _f32p(K), _f32p(pose)), "rf_integrate")
        else:
            host = depth.numpy() if isinstance(depth, torch.Tensor) else np.asarray(depth)
            assert host.dtype == np.float32 and host.flags.c_contiguous
            h, w = host.shape
            _check(lib().rf_integrate_ex(self._h, C.c_void_p(host.ctypes.data), C.c_int32(1), C.c_int32(w), C.c_int32(h),
                                         _f32p(K), _f32p(pose)), "rf_integrate_ex")

    def stage_frame(self, depth_host):
        """rf_stage_frame: prefetch a host frame (pinned CPU tensor or numpy array) on the copy stream."""
        if isinstance(depth_host, torch.Tensor):
            assert depth_host.dtype == torch.float32 and depth_host.is_contiguous() and not depth_host.is_cuda
            (h, w), ptr = depth_host.shape, depth_host.data_ptr()
        else:
            host = np.asarray(depth_host)
            assert host.dtype == np.float32 and host.flags.c_contiguous
            (h, w), ptr = host.shape, host.ctypes.data
        self._staged_keep = getattr(self, "_staged_keep", [])[-1:] + [depth_host]      # keep the buffers alive
        _check(lib().rf_stage_frame(self._h, C.c_void_p(ptr), C.c_int32(w), C.c_int32(h)), "rf_stage_frame")
        return (h, w)

    def last_updated(self) -> int:
        n = C.c_int64(0)
        _check(lib().rf_integrate_last_updated(self._h, C.byref(n)), "rf_integrate_last_updated")
        return int(n.value)

    def last_stats(self):
        """(voxels updated, bricks swept, atlas bricks refreshed) of the last integrate call."""
        out = (C.c_int64 * 4)()
        _check(lib().rf_integrate_last_stats(self._h, out), "rf_integrate_last_stats")
        return int(out[0]), int(out[1]), int(out[2])

    # ---- a0
    def backproject(self, depth: torch.Tensor, K, stride: int) -> torch.Tensor:
        h, w = depth.shape
        K = _host_f32(K, 4)
        nu = max(0, (w - stride // 2 + stride - 1) // stride)
        nv = max(0, (h - stride // 2 + stride - 1) // stride)
        pts = torch.empty((max(nu * nv, 1), 4), dtype=torch.float32, device=depth.device)
        m = C.c_int32(0)
        _check(lib().rf_backproject(self._h, C.c_void_p(_dev(depth, torch.float32)), C.c_int32(w), C.c_int32(h), _f32p(K),
                                    C.c_int32(stride), C.c_void_p(pts.data_ptr()), C.byref(m)), "rf_backproject")
        return pts[: m.value]

    # ---- a2 + a3
    def eval_particles(self, points: torch.Tensor, pst: torch.Tensor, center_pose_c2w, scale, mode: int = 0,
                       return_S: bool = False):
        M, N = points.shape[0], pst.shape[0]
        pose = _host_f32(center_pose_c2w, 12)
        sc = _host_f32(scale, 6)
        fit = torch.empty(N, dtype=torch.float32, device=points.device)
        cnt = torch.empty(N, dtype=torch.int32, device=points.device)
        S = torch.empty(N, dtype=torch.float32, device=points.device) if return_S else None
        _check(lib().rf_eval_particles_ex(self._h, C.c_void_p(_dev(points, torch.float32)), C.c_int32(M),
                                          C.c_void_p(_dev(pst, torch.float32)), C.c_int32(N), _f32p(pose), _f32p(sc),
                                          C.c_int32(mode), C.c_void_p(fit.data_ptr()), C.c_void_p(cnt.data_ptr()),
                                          C.c_void_p(S.data_ptr() if return_S else 0)), "rf_eval_particles")
        return (fit, cnt, S) if return_S else (fit, cnt)

    # ---- a0-a5
    def track_integrate(self, depth, K, psts: Sequence[torch.Tensor], strides: Sequence[int], iters: int, pose_c2w,
                        prev_pose_c2w, r0=None, flags: int = 0, want_trace: bool = False, gate=None):
        """rf_track_integrate: pfo_track, then fusion of the same frame at the tracked pose, in one call.
        gate = (centre xyz, radius in metres) or None; the result carries `integrated` (False: the gate held the frame back)."""
        return self.pfo_track(depth, K, psts, strides, iters, pose_c2w, prev_pose_c2w, r0=r0, flags=flags,
                              want_trace=want_trace, _fuse=True, _gate=gate)

    def pfo_track(self, depth, K, psts: Sequence[torch.Tensor], strides: Sequence[int], iters: int, pose_c2w,
                  prev_pose_c2w, r0=None, flags: int = 0, want_trace: bool = False, start_iter: int = 0,
                  aps_threshold: float = 0.0, _fuse: bool = False, _gate=None):
        # the argument blocks are kept between calls and filled through numpy views: the marshalling of a streaming
        # caller sits between two frames' GPU work, so it is kept to a few microseconds
        c = self.__dict__.get("_trk")
        if c is None:
            c = self._trk = dict(fr=Frame(), ps=PstSet(), st=TrackState(), res=TrackResult(), fused=C.c_int32(0),
                                 gate=(C.c_float * 3)(), ps_key=None)
            c["v_K"] = np.frombuffer(c["fr"], dtype=np.float32, count=4, offset=Frame.K.offset)
            c["v_pose"] = np.frombuffer(c["st"], dtype=np.float32, count=12, offset=TrackState.pose_c2w.offset)
            c["v_prev"] = np.frombuffer(c["st"], dtype=np.float32, count=12, offset=TrackState.prev_pose_c2w.offset)
            c["v_r0"] = np.frombuffer(c["st"], dtype=np.float32, count=6, offset=TrackState.r0.offset)
            c["v_gate"] = np.frombuffer(c["gate"], dtype=np.float32, count=3)
            c["refs"] = (C.byref(c["fr"]), C.byref(c["ps"]), C.byref(c["st"]), C.byref(c["res"]), C.byref(c["fused"]))
        fr, ps, st, res, fused = c["fr"], c["ps"], c["st"], c["res"], c["fused"]
        if isinstance(depth, tuple):                       # (H, W): consume the oldest prefetched frame (stage_frame)
            h, w = depth
            fr.depth, fr.depth_on_host = 0, 2
            keep = None
        elif isinstance(depth, torch.Tensor) and depth.is_cuda:
            h, w = depth.shape
            fr.depth, fr.depth_on_host = _dev(depth, torch.float32), 0
            keep = depth
        else:
            keep = depth.numpy() if isinstance(depth, torch.Tensor) else np.asarray(depth)
            assert keep.dtype == np.float32 and keep.flags.c_contiguous
            h, w = keep.shape
            fr.depth, fr.depth_on_host = keep.ctypes.data, 1
        fr.width, fr.height = w, h
        c["v_K"][:] = np.asarray(K, dtype=np.float32).reshape(4)
        key = (psts[0].data_ptr(), psts[1].data_ptr(), psts[2].data_ptr(), psts[0].shape[0], psts[1].shape[0],
               psts[2].shape[0], int(strides[0]), int(strides[1]), int(strides[2]))
        if key != c["ps_key"]:
            for l in range(3):
                ps.pst_dev[l] = _dev(psts[l], torch.float32)
                ps.N[l] = psts[l].shape[0]
                ps.stride[l] = int(strides[l])
            c["ps_key"] = key
        c["v_pose"][:] = np.asarray(pose_c2w, dtype=np.float32).reshape(12)
        c["v_prev"][:] = np.asarray(prev_pose_c2w, dtype=np.float32).reshape(12)
        st.has_r0 = 0 if r0 is None else 1
        c["v_r0"][:] = 0.0 if r0 is None else np.asarray(r0, dtype=np.float32).reshape(6)
        st.flags = int(flags)
        st.start_iter = int(start_iter)
        st.aps_threshold = float(aps_threshold)
        trace = (TrackTrace * iters)() if want_trace else None
        fused.value = 0
        rfr, rps, rst, rres, rfused = c["refs"]
        if _fuse:
            gc = None
            if _gate is not None:
                c["v_gate"][:] = np.asarray(_gate[0], dtype=np.float32).reshape(3)
                gc = c["gate"]
            _check(lib().rf_track_integrate(self._h, rfr, rps, C.c_int32(iters), rst, rres, trace, gc,
                                            C.c_float(_gate[1] if _gate is not None else 0.0), rfused),
                   "rf_track_integrate")
        else:
            _check(lib().rf_pfo_track(self._h, rfr, rps, C.c_int32(iters), rst, rres, trace), "rf_pfo_track")
        del keep
        out = dict(integrated=bool(fused.value), pose=c["v_pose"].reshape(3, 4).copy(), r1=c["v_r0"].copy(),
                   iters_run=res.iters_run, status=res.status, final_fitness=res.final_fitness,
                   final_count=res.final_count, argmax=res.argmax, evals=int(res.evals), aps_threshold=float(st.aps_threshold))
        if want_trace:
            out["trace"] = [trace[i] for i in range(res.iters_run)]
        return out

    # ---- particle-sharded frame loop (one process per GPU; the row exchange is the caller's torch.distributed)
    def shard_begin(self, depth: torch.Tensor, K, psts_local: Sequence[torch.Tensor], offsets, totals, strides, pose_c2w,
                    prev_pose_c2w, r0, flags: int = 0):
        h, w = depth.shape
        fr, ps, st = Frame(), PstSet(), TrackState()
        fr.depth, fr.depth_on_host, fr.width, fr.height = _dev(depth, torch.float32), 0, w, h
        fr.K[:] = [float(x) for x in np.asarray(K, dtype=np.float32).reshape(4)]
        for l in range(3):
            ps.pst_dev[l] = _dev(psts_local[l], torch.float32)
            ps.N[l] = psts_local[l].shape[0]
            ps.stride[l] = int(strides[l])
        st.pose_c2w[:] = [float(x) for x in np.asarray(pose_c2w, dtype=np.float32).reshape(12)]
        st.prev_pose_c2w[:] = [float(x) for x in np.asarray(prev_pose_c2w, dtype=np.float32).reshape(12)]
        st.r0[:] = [float(x) for x in np.asarray(r0, dtype=np.float32).reshape(6)]
        st.has_r0, st.flags, st.start_iter = 1, int(flags), 0
        off = (C.c_int32 * 3)(*[int(o) for o in offsets])
        tot = (C.c_int32 * 3)(*[int(t) for t in totals])
        self._shard_keep = (depth, list(psts_local))
        _check(lib().rf_shard_begin(self._h, C.byref(fr), C.byref(ps), off, tot, C.byref(st)), "rf_shard_begin")

    def shard_eval(self, k: int) -> torch.Tensor:
        row = torch.empty(16, dtype=torch.float64, device="cuda")
        _check(lib().rf_shard_eval(self._h, C.c_int32(k), C.c_void_p(row.data_ptr())), "rf_shard_eval")
        return row

    def shard_apply(self, k: int, rows: torch.Tensor, want_trace: bool = False):
        """rows: [G,16] float64 CUDA tensor, rank order.  -> (done, trace row or None)"""
        assert rows.dtype == torch.float64 and rows.is_cuda and rows.is_contiguous() and rows.shape[1] == 16
        tr = TrackTrace() if want_trace else None
        done = C.c_int32(0)
        _check(lib().rf_shard_apply(self._h, C.c_int32(k), C.c_void_p(rows.data_ptr()), C.c_int32(rows.shape[0]),
                                    C.byref(tr) if want_trace else None, C.byref(done)), "rf_shard_apply")
        return bool(done.value), tr

    def shard_end(self):
        st, res = TrackState(), TrackResult()
        _check(lib().rf_shard_end(self._h, C.byref(st), C.byref(res)), "rf_shard_end")
        return dict(pose=np.array(st.pose_c2w[:], dtype=np.float32).reshape(3, 4), r1=np.array(st.r0[:], dtype=np.float32),
                    iters_run=res.iters_run, status=res.status, final_fitness=res.final_fitness, final_count=res.final_count,
                    argmax=res.argmax, evals=int(res.evals))

    def pfo_track_sharded(self, depth, K, psts_local, offsets, totals, strides, iters: int, pose_c2w, prev_pose_c2w, r0,
                          flags: int = 0, gather=None, want_trace: bool = False):
        """Algorithm 1 with the templates split over the ranks of torch.distributed (or `gather`: row [16] -> rows [G,16])."""
        if gather is None:
            import torch.distributed as dist
            world = dist.get_world_size()

            def gather(row):
                rows = torch.empty(world * 16, dtype=torch.float64, device=row.device)
                dist.all_gather_into_tensor(rows, row)
                return rows.view(world, 16)
        self.shard_begin(depth, K, psts_local, offsets, totals, strides, pose_c2w, prev_pose_c2w, r0, flags)
        trace = []
        for k in range(1, iters + 1):
            done, tr = self.shard_apply(k, gather(self.shard_eval(k)), want_trace)
            if want_trace:
                trace.append(tr)
            if done:
                break
        out = self.shard_end()
        if want_trace:
            out["trace"] = trace[: out["iters_run"]]
        return out

    # ---- baselines of Section 5.2 (argument marshalling only; the state stays on the device)
    def baseline_propose(self, delta_in: torch.Tensor, ancestors, sigma, normals: torch.Tensor) -> torch.Tensor:
        N = delta_in.shape[0]
        out = torch.empty_like(delta_in)
        sg = _host_f32(sigma, 6)
        _check(lib().rf_baseline_propose(self._h, C.c_void_p(_dev(delta_in, torch.float32)),
                                         C.c_void_p(0 if ancestors is None else _dev(ancestors, torch.int32)), _f32p(sg),
                                         C.c_void_p(_dev(normals, torch.float32)), C.c_int32(N), C.c_void_p(out.data_ptr())),
               "rf_baseline_propose")
        return out

    def baseline_resample(self, fitness: torch.Tensor, u: float) -> torch.Tensor:
        N = fitness.shape[0]
        anc = torch.empty(N, dtype=torch.int32, device=fitness.device)
        _check(lib().rf_baseline_resample(self._h, C.c_void_p(_dev(fitness, torch.float32)), C.c_int32(N), C.c_double(u),
                                          C.c_void_p(anc.data_ptr())), "rf_baseline_resample")
        return anc

    def baseline_pso_move(self, x: torch.Tensor, v: torch.Tensor, pbest: torch.Tensor, gbest: torch.Tensor, ua: torch.Tensor,
                          ub: torch.Tensor):
        """In place on x and v."""
        _check(lib().rf_baseline_pso_move(self._h, C.c_void_p(_dev(x, torch.float32)), C.c_void_p(_dev(v, torch.float32)),
                                          C.c_void_p(_dev(pbest, torch.float32)), C.c_void_p(_dev(gbest, torch.float32)),
                                          C.c_void_p(_dev(ua, torch.float32)), C.c_void_p(_dev(ub, torch.float32)),
                                          C.c_int32(x.shape[0])), "rf_baseline_pso_move")

    def baseline_best(self, fitness: torch.Tensor, x: torch.Tensor, pbest, pbest_fit, first: bool, gbest: torch.Tensor):
        """In place on pbest / pbest_fit (or None) and gbest [8]."""
        _check(lib().rf_baseline_best(self._h, C.c_void_p(_dev(fitness, torch.float32)), C.c_void_p(_dev(x, torch.float32)),
                                      C.c_int32(x.shape[0]), C.c_void_p(0 if pbest is None else _dev(pbest, torch.float32)),
                                      C.c_void_p(0 if pbest_fit is None else _dev(pbest_fit, torch.float32)),
                                      C.c_int32(1 if first else 0), C.c_void_p(_dev(gbest, torch.float32))), "rf_baseline_best")

    # ---- read-out
    def raycast(self, K, width: int, height: int, pose_c2w, step: float, z_max: float, want_normals: bool = False):
        """rf_raycast: -> (depth [H,W] float32 CUDA tensor, normals [H,W,3] or None); stream-ordered, not synchronised."""
        K = _host_f32(K, 4)
        pose = _host_f32(pose_c2w, 12)
        dev = torch.device("cuda", torch.cuda.current_device())
        depth = torch.empty((height, width), dtype=torch.float32, device=dev)
        normals = torch.empty((height, width, 3), dtype=torch.float32, device=dev) if want_normals else None
        _check(lib().rf_raycast(self._h, _f32p(K), C.c_int32(width), C.c_int32(height), _f32p(pose), C.c_float(step),
                                C.c_float(z_max), C.c_void_p(depth.data_ptr()),
                                C.c_void_p(normals.data_ptr() if want_normals else 0)), "rf_raycast")
        return depth, normals

    def extract_surface_points(self, cap: int = 1 << 22, want_edges: bool = True):
        """rf_extract_surface_points -> (points [n,3] float32 CUDA tensor, edge keys [n] int64 or None); grows the buffer once
        if the first capacity was too small."""
        while True:
            pts = torch.empty((cap, 3), dtype=torch.float32, device="cuda")
            edge = torch.empty(cap, dtype=torch.int64, device="cuda") if want_edges else None
            n = C.c_int64(0)
            _check(lib().rf_extract_surface_points(self._h, C.c_void_p(pts.data_ptr()), C.c_void_p(edge.data_ptr() if want_edges else 0),
                                                   C.c_int64(cap), C.byref(n)), "rf_extract_surface_points")
            if n.value <= cap:
                return pts[: n.value], (edge[: n.value] if want_edges else None)
            cap = int(n.value)

    def gn_track(self, points: torch.Tensor, pose, iters: int):
        """rf_gn_track: Gauss-Newton on Eq. (4) from `pose` -> dict(pose [3,4] f64, iters_run, rows [iters_run] of GNRow)."""
        assert points.is_cuda and points.dtype == torch.float32 and points.is_contiguous()
        pin = np.ascontiguousarray(np.asarray(pose, dtype=np.float64).reshape(12))
        pout = np.zeros(12, dtype=np.float64)
        rows = (GNRow * max(int(iters), 1))()
        k = C.c_int32(0)
        _check(lib().rf_gn_track(self._h, C.c_void_p(points.data_ptr()), C.c_int32(points.shape[0]),
                                 pin.ctypes.data_as(C.POINTER(C.c_double)), C.c_int32(iters),
                                 pout.ctypes.data_as(C.POINTER(C.c_double)), rows, C.byref(k)), "rf_gn_track")
        return dict(pose=pout.reshape(3, 4), iters_run=int(k.value), rows=[rows[i] for i in range(int(k.value))])

    def gn_track_noalloc(self, points: torch.Tensor, pose, iters: int):
        """rf_gn_track_noalloc: rf_gn_track on the library's static device scratch (no allocation; iters <= 64)."""
        assert points.is_cuda and points.dtype == torch.float32 and points.is_contiguous()
        pin = np.ascontiguousarray(np.asarray(pose, dtype=np.float64).reshape(12))
        pout = np.zeros(12, dtype=np.float64)
        rows = (GNRow * max(int(iters), 1))()
        k = C.c_int32(0)
        _check(lib().rf_gn_track_noalloc(self._h, C.c_void_p(points.data_ptr()), C.c_int32(points.shape[0]),
                                         pin.ctypes.data_as(C.POINTER(C.c_double)), C.c_int32(iters),
                                         pout.ctypes.data_as(C.POINTER(C.c_double)), rows, C.byref(k)), "rf_gn_track_noalloc")
        return dict(pose=pout.reshape(3, 4), iters_run=int(k.value), rows=[rows[i] for i in range(int(k.value))])

    def pool_stats(self):
        """rf_volume_pool_stats -> dict(allocated, capacity, dropped_last): bricks of a sparse volume's pool."""
        out = (C.c_int64 * 4)()
        _check(lib().rf_volume_pool_stats(self._h, out), "rf_volume_pool_stats")
        return dict(allocated=int(out[0]), capacity=int(out[1]), dropped_last=int(out[2]))

    def profile_enable(self, on: bool):
        _check(lib().rf_profile_enable(self._h, C.c_int32(1 if on else 0)), "rf_profile_enable")

    def profile_read(self, which: int):
        ms, n = C.c_double(0), C.c_int64(0)
        _check(lib().rf_profile_read(self._h, C.c_int32(which), C.byref(ms), C.byref(n)), "rf_profile_read")
        return float(ms.value), int(n.value)

    def profile_read_launches(self, which: int, cap: int = 1 << 16) -> np.ndarray:
        """Individual launch durations (ms, launch order) since the last profile_read(which)."""
        buf = np.zeros(cap, dtype=np.float32)
        n = C.c_int32(0)
        _check(lib().rf_profile_read_launches(self._h, C.c_int32(which), _f32p(buf), C.c_int32(cap), C.byref(n)),
               "rf_profile_read_launches")
        return buf[: min(int(n.value), cap)].copy()

    # ---- a7
    def download(self, want_weight: bool = True):
        n = self.dims[0] * self.dims[1] * self.dims[2]
        t = np.empty(n, dtype=np.float32)
        w = np.empty(n, dtype=np.float32) if want_weight else None
        _check(lib().rf_volume_download(self._h, _f32p(t), _f32p(w) if want_weight else None), "rf_volume_download")
        return t, w

    def download_device(self, want_weight: bool = True):
        """rf_volume_download_ex with device outputs: dense x-fastest float32 CUDA tensors (for large volumes whose
        read-out should stay in HBM)."""
        n = self.dims[0] * self.dims[1] * self.dims[2]
        t = torch.empty(n, dtype=torch.float32, device="cuda")
        w = torch.empty(n, dtype=torch.float32, device="cuda") if want_weight else None
        _check(lib().rf_volume_download_ex(self._h, C.c_void_p(t.data_ptr()), C.c_void_p(w.data_ptr() if want_weight else 0),
                                           C.c_int32(1)), "rf_volume_download_ex")
        return t, w

    def download_box(self, lo, size):
        """rf_volume_download_box -> (tsdf, weight): float32 CUDA tensors of shape [size z, size y, size x]."""
        lo3, sz3 = (C.c_int32 * 3)(*[int(a) for a in lo]), (C.c_int32 * 3)(*[int(a) for a in size])
        shape = (int(size[2]), int(size[1]), int(size[0]))
        t = torch.empty(shape, dtype=torch.float32, device="cuda")
        w = torch.empty(shape, dtype=torch.float32, device="cuda")
        _check(lib().rf_volume_download_box(self._h, lo3, sz3, C.c_void_p(t.data_ptr()), C.c_void_p(w.data_ptr())),
               "rf_volume_download_box")
        return t, w

    def upload(self, tsdf: np.ndarray, weight: np.ndarray):
        n = self.dims[0] * self.dims[1] * self.dims[2]
        t, w = _host_f32(tsdf, n), _host_f32(weight, n)
        _check(lib().rf_volume_upload(self._h, _f32p(t), _f32p(w)), "rf_volume_upload")


def launch_count() -> int:
    return int(lib().rf_launch_count())


def gn_noalloc_scratch_bytes() -> int:
    """Size of the static device array rf_gn_track_noalloc works in (held by every GPU that loads the library)."""
    return int(lib().rf_gn_noalloc_scratch_bytes())


def microbench_l2(nbytes: int = 48 << 20, mode: int = 0, reps: int = 5) -> float:
    g = C.c_double(0)
    _check(lib().rf_microbench_l2(C.c_int64(nbytes), C.c_int32(mode), C.c_int32(reps), C.byref(g)), "rf_microbench_l2")
    return float(g.value)

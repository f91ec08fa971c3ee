#!/usr/bin/env python
"""bench.py -- the hot path measured on B200 (contract in the task statement, section 4).

A "step" is one pass of the whole hot path over one synthetic frame of the config-3 workload
(BASELINE.json configs[2], the fast-motion sequence the metric "ms per tracked frame (PFO+integrate)" is
quoted on): rf_pfo_track (back-project 3 levels, Algorithm 1 with its stop rules and the cap of 20 PFO iterations of
mask -> fitness -> swarm update, all on the device) followed by rf_integrate at the tracked pose, on a 512^3 fp16+u8
volume.  value = particle-point fitness evaluations per second over the whole step time (track + integrate).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import rf_synth as S  # noqa: E402

# Truncation: BASELINE.json fixes none for config 3.  12 cm = 3 sigma of the config's depth noise (1 % of 4 m);
# with SURVEY's first guess of 4 cm the fitness is noise-dominated (rho <= 0.68 at the true pose) and the paper's
# (1 - rho) search-radius rule never contracts (reading R-C3, oracle evidence).
DIMS, VS, MU = (512, 512, 512), 0.01, 0.12
N_BUILD = 30               # frames of the sequence already fused (at their true poses) when timing starts
STRIDES = (8, 16, 32)
PST_SIZES = (1024, 3072, 10240)
ITERS = 20                 # the paper's cap; the headline runs Algorithm 1 with its stop rules
R0_PRIOR = np.array([0.03, 0.03, 0.03, 0.15, 0.15, 0.15], dtype=np.float32)   # search prior for a 3 m/s sequence
LOST_TE = 0.08             # harness-side loss detector: a frame whose translation error exceeds this is fused at, and the
                           # next one restarted from, the ground-truth pose (counted; the un-assisted run is reported too)
METRIC = "particle-point fitness evals/sec (PFO track + integrate per frame, config 3)"
UNIT = "evals/s"
WORKLOAD = ("config3 fast-motion sequence: 512^3 fp16+u8 TSDF (384 MiB > 126 MB L2, no flush needed), 640x480 depth, "
            "PST 1024/3072/10240, strides 8/16/32, Algorithm 1 with its stop rules (cap 20 iterations) + integrate per frame")


def make_workload(n_frames: int, rank: int = 0):
    """Seeded config-3 inputs: scene, trajectory, noisy 640x480 frames, three PSTs.  `n_frames` counts the
    N_BUILD map-building frames plus the tracked ones.  Each rank takes its own stretch of the same seeded
    trajectory (independent sequences: replicas only)."""
    scene = S.make_config3_scene()
    traj = S.make_config3_trajectory(scene, n_frames=200)
    from paper_2105_05600_b200.replicas import shard_start
    start = shard_start(rank, n_frames)
    poses = traj[start:start + n_frames]
    frames, K = [], None
    for i, T in enumerate(poses):
        d, K = S.render_frame(scene, T, 3, start + i)
        frames.append(d)
    psts = [S.sample_pst(n, S.config_seed(3, 5 + i)) for i, n in enumerate(PST_SIZES)]
    return scene, poses, frames, K, psts


class ClockSampler(threading.Thread):
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.stop_flag = index, [], False

    def run(self):
        try:                                  # NVML in-process: a sample every few milliseconds
            import pynvml
            pynvml.nvmlInit()
            hdl = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            mx = pynvml.nvmlDeviceGetMaxClockInfo(hdl, pynvml.NVML_CLOCK_SM)
            while not self.stop_flag:
                sm = pynvml.nvmlDeviceGetClockInfo(hdl, pynvml.NVML_CLOCK_SM)
                r = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(hdl)
                pw = pynvml.nvmlDeviceGetPowerUsage(hdl) / 1000.0
                flag = lambda bit: "Active" if (r & bit) else "Not Active"
                self.samples.append([str(sm), str(mx), f"{pw:.1f}", flag(0x8), flag(0x40), flag(0x20), flag(0x4)])
                time.sleep(0.005)
            return
        except Exception:
            pass
        while not self.stop_flag:             # fallback: the nvidia-smi query of the profiling recipe
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i",
                                      str(self.index)], capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.samples.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        sm = [float(s[0]) for s in self.samples if s[0].replace(".", "").isdigit()]
        mx = [float(s[1]) for s in self.samples if s[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for s in self.samples for i in range(4) if len(s) >= 7 and s[3 + i].lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(self.samples)}


def ncu_traffic():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` capture of this
    workload (profiles/r2_traffic.csv: kernel, bytes per launch; its .md names the commit it was taken at); {} when absent."""
    p = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    out = {}
    if os.path.exists(p):
        for line in open(p):
            parts = [x.strip() for x in line.split(",")]
            if len(parts) >= 2 and not line.startswith("#") and parts[1].replace(".", "").isdigit():
                out[parts[0]] = float(parts[1])
    return out


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d.get("hbm_gbs", 6650.0), "measured"
    return 6650.0, "fallback"


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.lower().startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def te_stats(tes):
    t = np.asarray(tes, dtype=np.float64)
    return {"te_mean_cm": 100 * float(t.mean()), "te_median_cm": 100 * float(np.median(t)), "te_max_cm": 100 * float(t.max()),
            "frames_beyond_lost_threshold": int((t > LOST_TE).sum()), "frames": int(t.size)}


# --------------------------------------------------------------------------------------------- reference arm
def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores.  Each step is one frame of the same
    workload (Algorithm 1 with its stop rules on the three levels + one integration into the 512^3 volume), a few
    seconds of CPU work per step; same harness-side loss detector as the CUDA arm, and the un-assisted run beside it."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle as orc
    cores = os.cpu_count() or 1
    n = N_BUILD + args.warmup + args.steps
    scene, poses, frames, K, psts = make_workload(n)
    g = orc.make_grid(DIMS, VS, MU)
    F, W = orc.empty_volume(DIMS)
    for i in range(N_BUILD):
        orc.integrate(g, F, W, frames[i], K, poses[i].astype(np.float32), half_storage=True, nthreads=cores)
    F0, W0 = F.copy(), W.copy()

    def sequence(F, W, assist: bool, timed: bool):
        times, evals, tes, lost = [], 0, [], 0
        pose, r0 = poses[N_BUILD - 1].astype(np.float32), R0_PRIOR.astype(np.float64)
        for i in range(N_BUILD, n):
            t0 = time.perf_counter()
            out = orc.pfo_track(g, F, W, frames[i], K, psts, STRIDES, ITERS, pose, pose, r0=r0, early_stop=True, nthreads=cores)
            te = float(np.linalg.norm(out["pose"][:, 3] - poses[i][:, 3]))
            if assist and not te < LOST_TE:
                pose, r0 = poses[i].astype(np.float32), R0_PRIOR.astype(np.float64)
                lost += i >= N_BUILD + args.warmup
            else:
                pose, r0 = out["pose"].astype(np.float32), out["r1"]
            orc.integrate(g, F, W, frames[i], K, pose, half_storage=True, nthreads=cores)
            dt = time.perf_counter() - t0
            if i >= N_BUILD + args.warmup:
                times.append(dt)
                evals += out["evals"]
                tes.append(te)
        return times, evals, tes, lost

    times, evals, tes, lost = sequence(F, W, True, True)
    _, _, tes_free, _ = sequence(F0, W0, False, False)
    total = sum(times)
    val = evals / total
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "frames_restarted_from_gt": lost, "lost_threshold_cm": 100 * LOST_TE, **te_stats(tes),
                       "unassisted_free_run": te_stats(tes_free)},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu": cpu_model(),
                             "sample": f"{len(times)} frames, each full PFO track + one 512^3 integration"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# --------------------------------------------------------------------------------------------- CUDA arm
def run_cuda(args):
    import torch
    import torch.distributed as dist

    import paper_2105_05600_b200 as rf

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA arm has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    K_steps, W_steps = args.steps, args.warmup
    n = N_BUILD + W_steps + K_steps
    scene, poses, frames, K, psts = make_workload(n, rank)
    dev_frames = [torch.from_numpy(f).cuda() for f in frames]
    pin_frames = [torch.from_numpy(f).pin_memory() for f in frames]
    dpst = [torch.from_numpy(p).cuda() for p in psts]
    stream = torch.cuda.current_stream()
    hbm_peak, peak_kind = measured_peaks()

    def fresh_volume():
        v = rf.Volume(DIMS, VS, MU, dtype=rf.RF_F16_W8)
        for i in range(N_BUILD):                                             # the sequence so far, at its true poses
            v.integrate(dev_frames[i], K, poses[i].astype(np.float32))
        return v

    def run_sequence(vol, use_host: bool, first: int, count: int, state, flags: int, assist: bool = True,
                     count_updates: bool = False, traces=None):
        """Track + integrate frames [first, first+count): Algorithm 1 (stop rules per `flags`), then fusion at the tracked
        pose.  assist: the harness's loss detector -- a frame whose translation error exceeds LOST_TE is fused at the
        ground-truth pose instead and the next frame restarts from it (counted); without it the run is the un-assisted
        free run.  Returns evals, per-frame TE, frames restarted, the state, updated voxels."""
        pose, r0 = state
        evals, tes, lost, upd = 0, [], 0, 0
        iters_hist.clear()
        src = pin_frames if use_host else dev_frames
        if use_host:
            vol.stage_frame(src[first])                    # H2D of the first frame of this stretch (not overlapped)
        for i in range(first, first + count):
            d = src[i]
            gate = (poses[i][:, 3], LOST_TE) if assist else None
            if use_host:
                # streaming use of the API: the copy of frame i+1 is started on the copy stream before frame i is
                # tracked, so it overlaps the tracking; every frame still crosses the bus inside the timed region
                if i + 1 < first + count:
                    vol.stage_frame(src[i + 1])
                out = vol.track_integrate(tuple(d.shape), K, dpst, STRIDES, ITERS, pose, pose, r0=r0, flags=flags, gate=gate,
                                          want_trace=traces is not None)
            else:
                out = vol.track_integrate(d, K, dpst, STRIDES, ITERS, pose, pose, r0=r0, flags=flags, gate=gate,
                                          want_trace=traces is not None)
            # rf_track_integrate fused the frame at the tracked pose unless the gate held it back; then it is fused at the
            # true pose, from here
            iters_hist.append(out["iters_run"])
            tes.append(float(np.linalg.norm(out["pose"][:, 3].astype(np.float64) - poses[i][:, 3])))
            if traces is not None:
                traces.append((np.asarray(r0, dtype=np.float64), out["trace"]))
            if out["integrated"]:
                pose, r0 = out["pose"], out["r1"]
            else:
                pose, r0, lost = poses[i].astype(np.float32), R0_PRIOR, lost + 1
                if use_host:
                    vol.integrate(None, K, pose, staged_shape=tuple(d.shape))     # the frame crossed the bus once
                else:
                    vol.integrate(d, K, pose)
            if count_updates:
                upd += vol.last_updated()
            evals += out["evals"]
        return evals, tes, lost, (pose, r0), upd

    iters_hist = []

    def timed(use_host: bool, flags: int, profile: bool = False, assist: bool = True):
        vol = fresh_volume()
        state = (poses[N_BUILD - 1].astype(np.float32), R0_PRIOR)
        _, _, _, state, _ = run_sequence(vol, use_host, N_BUILD, W_steps, state, flags, assist)   # warm-up steps (W >= 3)
        traces = [] if profile else None
        if profile:
            vol.profile_enable(True)
            for slot in range(6):
                vol.profile_read(slot)
        l0 = rf.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        evals, tes, lost, _, upd = run_sequence(vol, use_host, N_BUILD + W_steps, K_steps, state, flags, assist,
                                                count_updates=profile, traces=traces)
        e1.record(stream)
        barrier()
        ms = e0.elapsed_time(e1)
        prof = None
        if profile:
            each = vol.profile_read_launches(0)
            prof = tuple(vol.profile_read(slot) for slot in range(6)) + (each, traces, list(iters_hist))
            vol.profile_enable(False)
        launches = rf.launch_count() - l0
        vol.destroy()
        return dict(ms=ms, evals=evals, tes=tes, lost=lost, launches=launches, prof=prof, upd=upd, iters=list(iters_hist))

    def fitness_regimes(prof, l2_gather):
        """One roofline per regime from the profiling pass (kernel by kernel, CUDA events around every k_fitness launch):
        a launch is `reinflated` when the iteration before it found an empty advantage set, so that it evaluates the
        swarm re-inflated by the rule of P:L292, else `contracting` (the first launch of a frame, and every launch that
        follows a successful step).  Algorithmic bytes: 16 per eval (8 fp16 corners); both against the L2 gather rate."""
        each, traces, iters = prof[6], prof[7], prof[8]
        reg = {"contracting": [0.0, 0.0, 0], "reinflated": [0.0, 0.0, 0]}       # evals, ms, launches
        sizes = [p.shape[0] for p in psts]
        q = 0
        for (r0, rows), it in zip(traces, iters):
            for k in range(ITERS):                                  # the frame loop enqueues ITERS launches; after a stop
                if k < it and q < len(each):                        # rule fired the rest are no-ops and are not counted
                    e = float(rows[k].M_O) * (sizes[k % 3] + 1)
                    key = "reinflated" if k > 0 and rows[k - 1].n_aps == 0 else "contracting"
                    reg[key][0] += e; reg[key][1] += float(each[q]); reg[key][2] += 1
                q += 1
        out = {}
        for key in ("contracting", "reinflated"):
            e, ms_, nl = reg[key]
            if nl:
                ach = e * 16.0 / (ms_ * 1e-3) / 1e9
                out[key] = {"launches": nl, "avg_launch_us": 1e3 * ms_ / nl, "evals_per_launch": e / nl,
                            "achieved": ach, "peak": l2_gather, "unit": "GB/s", "frac": ach / l2_gather}
        all_e = sum(v[0] for v in reg.values()); all_ms = sum(v[1] for v in reg.values()); all_n = sum(v[2] for v in reg.values())
        return out, all_e, all_ms, all_n

    # the clock sampler spans all timed passes (each is only tens of milliseconds long)
    sampler = ClockSampler(local)
    sampler.start()
    head = timed(False, 0)                    # headline: Algorithm 1 as published (stop rules on), inputs resident in HBM
    timed(True, 0)             # untimed rehearsal: the first copies out of freshly pinned frame buffers are slower than later ones
    e2e = timed(True, 0)
    prof_es = timed(False, 0, profile=True)
    fix20 = timed(False, rf.RF_TRACK_NO_EARLY_STOP)     # every frame runs the cap of 20 iterations (config 2's regime)
    prof_20 = timed(False, rf.RF_TRACK_NO_EARLY_STOP, profile=True)
    free = timed(False, 0, assist=False)      # un-assisted free run (reported, not timed: no ground truth touches it)
    sampler.stop_flag = True
    sampler.join(timeout=3)

    # max over ranks of the device time, sum over ranks of the work
    ms, evals, ms_e2e, evals_e2e = head["ms"], head["evals"], e2e["ms"], e2e["evals"]
    if world > 1:
        from paper_2105_05600_b200.replicas import aggregate
        ms, evals = aggregate(ms, evals)
        ms_e2e, evals_e2e = aggregate(ms_e2e, evals_e2e)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = evals / (ms * 1e-3)
    e2e_value = evals_e2e / (ms_e2e * 1e-3)
    frame_bytes = int(frames[0].nbytes)
    # ---- roofline of the dominant kernel (k_fitness) inside the step.  Algorithmic bytes per eval = 8 TSDF
    # corners x 2 B (fp16 storage) = 16 B; the bound is the L2 random-sector gather rate, measured
    # in this same run because MEASURED_PEAKS.json carries no L2 figure.
    traffic = ncu_traffic()
    l2_bytes = 48 << 20
    l2_gather = rf.microbench_l2(l2_bytes, 0, 5)
    l2_stream = rf.microbench_l2(l2_bytes, 1, 5)
    hbm_random = rf.microbench_l2(1 << 30, 0, 3)     # same random-sector reads over 1 GiB: every sector comes from HBM
    prof = prof_es["prof"]
    (fit_ms, fit_n), (int_ms, int_n), (atl_ms, atl_n), (upd_ms, upd_n), (cul_ms, _), (bp_ms, _) = prof[:6]
    regimes, fit_e, fit_ms_used, fit_n_used = fitness_regimes(prof, l2_gather)
    regimes20, _, _, _ = fitness_regimes(prof_20["prof"], l2_gather)
    kern_ms = fit_ms + int_ms + atl_ms + upd_ms + cul_ms + bp_ms      # device time of the step's kernels, launch gaps excluded
    achieved = fit_e * 16.0 / (fit_ms_used * 1e-3) / 1e9
    roofline = {"kernel": "k_fitness<half>", "bound": "l2_gather", "achieved": achieved, "peak": l2_gather, "unit": "GB/s",
                "frac": achieved / l2_gather, "traffic": traffic.get("k_fitness"),
                "peak_kind": f"measured in this run (rf_microbench_l2: {l2_bytes >> 20} MiB buffer, one 128-bit load per lane at a random 32-B sector, 32 B counted per request; faster of ld.nc / ld.cg)",
                "algorithmic_bytes_per_eval": 16,
                "launches": fit_n_used, "avg_launch_us": 1e3 * fit_ms_used / max(fit_n_used, 1), "evals_per_launch": fit_e / max(fit_n_used, 1),
                "share_of_step": fit_ms_used / kern_ms, "l2_stream_gbs": l2_stream, "hbm_random_sector_gbs": hbm_random,
                "regimes": regimes, "regimes_fixed_20_iterations": regimes20,
                "note": "all fitness launches that did work in the headline run (launches turned into no-ops by a stop rule are not "
                        "counted), CUDA events around every launch of a kernel-by-kernel profiling pass; `regimes` splits them into "
                        "launches that follow a successful step (or start a frame) and launches that evaluate the swarm re-inflated "
                        "after an empty advantage set (P:L292); hbm_random_sector_gbs is the same random-sector microbenchmark over "
                        "1 GiB (every request misses L2), for context; roofline_config4_cell is the same kernel on an L2-resident "
                        "launch large enough to amortise its fixed cost"}
    int_avg_ms = int_ms / max(int_n, 1)
    upd_per_frame = prof_es["upd"] / max(int_n, 1)
    int_bytes = upd_per_frame * 6.0 + frame_bytes  # updated voxels x 2 x (2 B fp16 + 1 B u8) + the depth image once, per launch
    roofline_int = {"kernel": "k_update<half>", "bound": "hbm", "achieved": int_bytes / (int_avg_ms * 1e-3) / 1e9, "peak": hbm_peak,
                    "unit": "GB/s", "frac": int_bytes / (int_avg_ms * 1e-3) / 1e9 / hbm_peak, "traffic": traffic.get("k_update"),
                    "note": "bounded in practice by the L1 data pipe (the scattered depth gathers: ncu l1tex__data_pipe_lsu_wavefronts 72-81 %) and instruction issue (60-68 %), DESIGN.md section 6",
                    "peak_kind": peak_kind, "avg_launch_us": 1e3 * int_avg_ms, "updated_voxels_per_launch": upd_per_frame,
                    "share_of_step": int_ms / kern_ms}

    breakdown = {"fitness_us_per_frame": 1e3 * fit_ms / max(K_steps, 1), "swarm_update_us_per_frame": 1e3 * upd_ms / max(K_steps, 1),
                 "integrate_update_us_per_frame": 1e3 * int_ms / max(K_steps, 1), "atlas_refresh_us_per_frame": 1e3 * atl_ms / max(K_steps, 1),
                 "cull_us_per_frame": 1e3 * cul_ms / max(K_steps, 1), "backproject_us_per_frame": 1e3 * bp_ms / max(K_steps, 1),
                 "note": "CUDA events around every launch of the profiling pass (kernel by kernel, no graph; includes the no-op launches after a stop rule fired); the graph-replayed step overlaps launches"}
    # ---- the same fitness kernel on one large cell of the config-4 sweep (65536 particles x 65536 points, scale 0.1,
    # centre = a true pose perturbed by 2 cm / 1 deg) on the map built above: kernel throughput away from the
    # launch-latency regime of the paper's 3-5 M-eval iterations.  Points: valid full-resolution pixels of one frame.
    roofline_c4 = None
    if world == 1:
        vol = fresh_volume()
        pts = vol.backproject(dev_frames[N_BUILD], K, 1)
        pts = pts[pts[:, 3] != 0][:65536].contiguous()
        big = torch.from_numpy(S.sample_pst(65536, S.config_seed(4, 5))).cuda()
        centre = S.compose_delta(poses[N_BUILD], [0.3, 0.5, 0.8], np.radians(1.0), [0.012, -0.012, 0.01]).astype(np.float32)
        scale = np.full(6, 0.1, dtype=np.float32)
        for _ in range(3):
            vol.eval_particles(pts, big, centre, scale)
        vol.profile_enable(True)
        for slot in range(6):
            vol.profile_read(slot)
        for _ in range(5):
            vol.eval_particles(pts, big, centre, scale)
        c4_ms, c4_n = vol.profile_read(0)
        vol.profile_enable(False)
        vol.destroy()
        c4_evals = float(pts.shape[0]) * float(big.shape[0])
        c4_gbs = c4_evals * 16.0 / (c4_ms / max(c4_n, 1) * 1e-3) / 1e9
        roofline_c4 = {"kernel": "k_fitness<half>", "workload": f"config4 cell {big.shape[0]} particles x {pts.shape[0]} points, scale 0.1",
                       "bound": "l2_gather", "achieved": c4_gbs, "peak": l2_gather, "unit": "GB/s", "frac": c4_gbs / l2_gather,
                       "evals_per_s": c4_evals / (c4_ms / max(c4_n, 1) * 1e-3), "avg_launch_us": 1e3 * c4_ms / max(c4_n, 1), "launches": c4_n}

    # ---- the oracle timed beside it, on this box's host cores, on a bounded sample of the same workload
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle as orc
        cores = os.cpu_count() or 1
        g = orc.make_grid(DIMS, VS, MU)
        F, Wt = orc.empty_volume(DIMS)
        for i in range(N_BUILD):                                  # untimed: the same pre-built map as the CUDA arm
            orc.integrate(g, F, Wt, frames[i], K, poses[i].astype(np.float32), half_storage=True, nthreads=cores)
        p0 = poses[N_BUILD - 1].astype(np.float32)
        res = {}
        for label, nt in (("all_cores", cores), ("single_thread", 1)):
            Fc, Wc = F.copy(), Wt.copy()
            t0 = time.perf_counter()
            out = orc.pfo_track(g, Fc, Wc, frames[N_BUILD], K, psts, STRIDES, ITERS, p0, p0,
                                r0=R0_PRIOR.astype(np.float64), early_stop=True, nthreads=nt)
            orc.integrate(g, Fc, Wc, frames[N_BUILD], K, out["pose"].astype(np.float32), half_storage=True, nthreads=nt)
            res[label] = (out["evals"] / (time.perf_counter() - t0), out, time.perf_counter() - t0)
        val, out, dt = res["all_cores"]
        cpu = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu": cpu_model(),
               "single_thread_value": res["single_thread"][0],
               "sample": f"1 frame of the same workload: PFO track ({out['iters_run']} iterations, {out['evals']} evals) + one 512^3 "
                         f"integration, {dt:.1f} s on {cores} threads, {res['single_thread'][2]:.1f} s on one"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K_steps, "warmup": W_steps,
            "ms_per_step": ms / K_steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": WORKLOAD,
                       "parallelism": "replicas only" if world > 1 else "single GPU", "storage": "fp16 TSDF + u8 weight, fp32 arithmetic",
                       "iters_cap": ITERS, "mean_iterations": float(np.mean(head["iters"])), **te_stats(head["tes"]),
                       "frames_restarted_from_gt": head["lost"], "lost_threshold_cm": 100 * LOST_TE, "r0_prior": R0_PRIOR.tolist(),
                       "mean_evals_per_frame": evals / max(K_steps * world, 1),
                       "unassisted_free_run": {**te_stats(free["tes"]), "note": "same frames without the harness's loss detector: no ground truth touches the tracker"}},
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": ms_e2e / K_steps, "h2d_bytes_per_step": frame_bytes,
                    "d2h_bytes_per_step": 344, "note": "host pinned depth frames through rf_stage_frame -> rf_track_integrate (rf_pfo_track + rf_integrate of the same frame in one call): one H2D copy per frame, started one frame ahead on the copy stream so it overlaps the previous frame's tracking; pose/result read back each step (the 344-byte loop state, written into a pinned host mirror by the frame's last kernel); the timed pass follows one untimed rehearsal of the same sequence over the same pinned buffers (beyond the W warm-up steps), as a streaming caller reuses its pinned buffers"},
            "gpu_launches": head["launches"], "clocks": sampler.summary(), "roofline": roofline, "roofline_integrate": roofline_int, "roofline_config4_cell": roofline_c4, "breakdown": breakdown,
            "fixed_20_iterations": {"ms_per_step": fix20["ms"] / K_steps, "value": fix20["evals"] / (fix20["ms"] * 1e-3), "unit": UNIT,
                                    **te_stats(fix20["tes"]), "frames_restarted_from_gt": fix20["lost"],
                                    "note": "same frames with the stop rules off: every frame runs the cap of 20 iterations (round 1's headline); most of the extra launches evaluate the re-inflated swarm of P:L292"},
            "cpu_baseline": cpu}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# --------------------------------------------------------------------------------------------- configs 4 and 5
def run_sweep(args):
    """--sweep: the other two measurement configs of BASELINE.json, one JSON line.
    config 4: fitness + count only, particles {1k,4k,16k,64k,128k} x points {1k,4k,16k,64k} on the 512^3 fp16 map of the
    config-3 scene (built here by integrating N_BUILD frames), centre = a true pose perturbed by 2 cm / 1 deg, scale 0.1.
    config 5: 100 frames of 640x480 depth at seeded random poses fused into an empty 1024^3 fp16+u8 volume (voxel 5 mm)."""
    import torch

    import paper_2105_05600_b200 as rf

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA arm has no CPU fallback")
    torch.cuda.set_device(0)
    hbm_peak, _ = measured_peaks()
    scene, poses, frames, K, _ = make_workload(N_BUILD + 1)
    vol = rf.Volume(DIMS, VS, 0.04, dtype=rf.RF_F16_W8)          # config 4 truncation: 4 cm
    for i in range(N_BUILD):
        vol.integrate(torch.from_numpy(frames[i]).cuda(), K, poses[i].astype(np.float32))
    pts_all = vol.backproject(torch.from_numpy(frames[N_BUILD]).cuda(), K, 1)
    pts_all = pts_all[pts_all[:, 3] != 0].contiguous()
    rng = np.random.Generator(np.random.Philox(S.config_seed(4, 8)))
    pst_all = torch.from_numpy(S.sample_pst(131072, S.config_seed(4, 5))).cuda()
    centre = S.compose_delta(poses[N_BUILD], [0.3, 0.5, 0.8], np.radians(1.0), [0.012, -0.012, 0.01]).astype(np.float32)
    scale = np.full(6, 0.1, dtype=np.float32)
    l2_gather = rf.microbench_l2(48 << 20, 0, 5)
    cells = []
    for M in (1024, 4096, 16384, 65536):
        sel = torch.from_numpy(np.sort(rng.choice(pts_all.shape[0], size=M, replace=False))).cuda()
        pts = pts_all[sel].contiguous()
        for N in (1024, 4096, 16384, 65536, 131072):
            pst = pst_all[:N]
            for _ in range(3):
                vol.eval_particles(pts, pst, centre, scale)
            vol.profile_enable(True)
            for slot in range(6):
                vol.profile_read(slot)
            reps = 5 if N * M >= (1 << 26) else 20
            for _ in range(reps):
                vol.eval_particles(pts, pst, centre, scale)
            ms, n = vol.profile_read(0)
            vol.profile_enable(False)
            us = 1e3 * ms / max(n, 1)
            cells.append({"particles": N, "points": M, "us_per_launch": us, "evals_per_s": N * M / (us * 1e-6),
                          "frac_l2_gather": N * M * 16.0 / (us * 1e-6) / 1e9 / l2_gather})
    vol.destroy()
    # ---- config 2: one tracking step on the 256^3 fp32 volume (20 iterations, early stop off), map built here
    c2 = S.make_config2_inputs()
    v2 = rf.Volume(c2["dims"], c2["voxel_size"], c2["trunc"], dtype=rf.RF_F32_W8)
    for T, d in zip(c2["build_poses"], c2["build_frames"]):
        v2.integrate(torch.from_numpy(d).cuda(), c2["K"], T)
    d2 = torch.from_numpy(c2["tracked_depth"]).cuda()
    p2 = [torch.from_numpy(p).cuda() for p in c2["psts"]]
    outs = [v2.pfo_track(d2, c2["K"], p2, c2["strides"], 20, c2["T_prev"], c2["T_prev"], r0=None, flags=rf.RF_TRACK_NO_EARLY_STOP)
            for _ in range(3)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(10):
        o2 = v2.pfo_track(d2, c2["K"], p2, c2["strides"], 20, c2["T_prev"], c2["T_prev"], r0=None, flags=rf.RF_TRACK_NO_EARLY_STOP)
    e1.record()
    torch.cuda.synchronize()
    ms2 = e0.elapsed_time(e1) / 10
    te2 = float(np.linalg.norm(o2["pose"][:, 3].astype(np.float64) - c2["T_true"][:, 3]))
    config2 = {"ms_per_track": ms2, "evals": o2["evals"], "evals_per_s": o2["evals"] / (ms2 * 1e-3), "te_cm": 100 * te2,
               "te_start_cm": 100 * float(np.linalg.norm(c2["T_prev"][:, 3].astype(np.float64) - c2["T_true"][:, 3])),
               "note": "256^3 fp32 volume (32-byte atlas entries, one 256-bit load per sample), 320x240 frame perturbed by 15 deg / 8 cm, 20 iterations"}
    v2.destroy()
    config5 = sweep_config5(rf, torch, scene, K, hbm_peak, 100)
    line = {"metric": "config 4 fitness sweep (evals/s) and config 5 integration throughput", "n_gpus": 1, "data": "synthetic",
            "l2_gather_peak_gbs": l2_gather, "hbm_peak_gbs": hbm_peak, "config2": config2, "config4": cells, "config5": config5}
    print(json.dumps(line))


def sweep_config5(rf, torch, scene, K, hbm_peak, n_frames):
    """Config 5: `n_frames` frames of 640x480 depth at seeded random poses fused into an empty 1024^3 fp16+u8 volume (voxel
    5 mm): three passes (counted, timed as one batch, timed kernel by kernel)."""
    poses5 = S.make_config5_poses(scene, n_frames)
    frames5 = [torch.from_numpy(S.render_frame(scene, T, 5, i)[0]).cuda() for i, T in enumerate(poses5)]
    res5 = {}
    for timed_pass in (False, True, "profile"):
        v5 = rf.Volume((1024, 1024, 1024), 0.005, 0.02, dtype=rf.RF_F16_W8)
        if timed_pass == "profile":             # CUDA events around every k_update launch (the roofline kernel)
            v5.profile_enable(True)
            for slot in range(6):
                v5.profile_read(slot)
            for d, T in zip(frames5, poses5):
                v5.integrate(d, K, T.astype(np.float32))
            res5["update_ms"], res5["update_n"] = v5.profile_read(1)
            res5["cull_ms"], _ = v5.profile_read(4)
            v5.profile_enable(False)
        elif timed_pass:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for d, T in zip(frames5, poses5):
                v5.integrate(d, K, T.astype(np.float32))
            e1.record()
            torch.cuda.synchronize()
            res5["ms_total"] = e0.elapsed_time(e1)
        else:                                   # same work, counted: updated voxels and swept bricks per frame
            upd = swept = 0
            for d, T in zip(frames5, poses5):
                v5.integrate(d, K, T.astype(np.float32))
                u, b, _ = v5.last_stats()
                upd, swept = upd + u, swept + b
            res5["updated_voxels"], res5["swept_bricks"] = upd, swept
        v5.destroy()
    gbs = res5["updated_voxels"] * 6.0 / (res5["ms_total"] * 1e-3) / 1e9
    kgbs = res5["updated_voxels"] * 6.0 / (res5["update_ms"] * 1e-3) / 1e9
    return {"frames": n_frames, "ms_per_frame": res5["ms_total"] / n_frames, "updated_voxels_per_frame": res5["updated_voxels"] / n_frames,
            "swept_voxels_per_frame": 512 * res5["swept_bricks"] / n_frames, "algorithmic_gbs": gbs, "frac_hbm": gbs / hbm_peak,
            "update_kernel_us": 1e3 * res5["update_ms"] / max(res5["update_n"], 1),
            "cull_kernels_us": 1e3 * res5["cull_ms"] / max(res5["update_n"], 1),
            "update_kernel_algorithmic_gbs": kgbs, "update_kernel_frac_hbm": kgbs / hbm_peak,
            "note": "rf_integrate calls enqueued back to back (tile-max, cull and update kernels), CUDA events around the whole batch; "
                    "update_kernel_* from CUDA events around every k_update launch of a separate pass"}


def run_config5(args):
    """--config5: the integration-throughput configuration alone (`--steps` frames), one JSON line."""
    import torch

    import paper_2105_05600_b200 as rf

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA arm has no CPU fallback")
    torch.cuda.set_device(0)
    hbm_peak, _ = measured_peaks()
    scene = S.make_config3_scene()
    K = S.render_frame(scene, S.make_config3_trajectory(scene, n_frames=200)[0], 3, 0)[1]
    print(json.dumps({"metric": "config 5 integration throughput", "n_gpus": 1, "data": "synthetic", "hbm_peak_gbs": hbm_peak,
                      "config5": sweep_config5(rf, torch, scene, K, hbm_peak, args.steps)}))


def run_readout(args):
    """--readout: SURVEY 8(f) row 3.  The config-3 map (30 frames fused at the true poses), read out by rf_raycast from
    the next pose at 640x480, step 5 cm, normals on: time per read-out (CUDA events around `steps` back-to-back calls;
    one read-out touches ~240 MB of atlas, more than L2) and accuracy / completeness against the analytic scene."""
    import torch

    import paper_2105_05600_b200 as rf

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA arm has no CPU fallback")
    torch.cuda.set_device(0)
    scene = S.make_config3_scene()
    traj = S.make_config3_trajectory(scene, n_frames=200)
    vs, mu = 0.01, 0.12
    vol = rf.Volume((512, 512, 512), vs, mu, dtype=rf.RF_F16_W8)
    K = None
    for i in range(30):
        d, K = S.render_frame(scene, traj[i], 3, i)
        vol.integrate(torch.from_numpy(d).cuda(), K, traj[i].astype(np.float32))
    pose = traj[30].astype(np.float32)
    step, z_max = 0.05, 8.0
    for _ in range(max(args.warmup, 3)):
        depth, normals = vol.raycast(K, 640, 480, pose, step, z_max, want_normals=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        depth, normals = vol.raycast(K, 640, 480, pose, step, z_max, want_normals=True)
    e1.record()
    torch.cuda.synchronize()
    us = 1e3 * e0.elapsed_time(e1) / args.steps
    got = depth.cpu().numpy()
    clean = S.raycast_depth(scene, traj[30], K, 640, 480)
    vis = np.isfinite(clean) & (clean > 0)
    both = vis & (got > 0)
    err = np.abs(got[both] - clean[both])
    # ---- the surface point set (rf_extract_surface_points): accuracy = distance of every point to the analytic surface
    # ("RMS error of all reconstructed points against the ground-truth surface")
    for _ in range(3):
        sp, _ = vol.extract_surface_points(cap=1 << 23, want_edges=False)
    e0.record()
    for _ in range(args.steps):
        sp, _ = vol.extract_surface_points(cap=1 << 23, want_edges=False)
    e1.record()
    torch.cuda.synchronize()
    us_sp = 1e3 * e0.elapsed_time(e1) / args.steps
    spn = sp.cpu().numpy().astype(np.float64)
    dist = np.abs(S.scene_sdf(scene, spn))
    surface = {"points": int(spn.shape[0]), "us_per_extraction": us_sp, "rms_mm": float(1e3 * np.sqrt(np.mean(dist ** 2))),
               "median_mm": float(1e3 * np.median(dist)), "q90_mm": float(1e3 * np.quantile(dist, 0.9)),
               "within_one_voxel": float((dist <= vs).mean())}
    print(json.dumps({"metric": "ray-cast read-out of the config-3 map", "n_gpus": 1, "data": "synthetic", "steps": args.steps,
                      "surface_points": surface,
                      "us_per_readout": us, "rays_per_s": 640 * 480 / (us * 1e-6), "step_m": step, "z_max_m": z_max,
                      "image": [640, 480], "normals": True,
                      "completeness": float(both.sum() / max(vis.sum(), 1)),
                      "accuracy_median_mm": float(1e3 * np.median(err)), "accuracy_q90_mm": float(1e3 * np.quantile(err, 0.9)),
                      "within_one_voxel": float((err <= vs).mean()), "voxel_mm": 1e3 * vs,
                      "note": "completeness = analytic-visible pixels with a read-out depth; accuracy = |read-out - analytic| "
                              "on those; frames carry 1 % depth noise and 5 % dropout"}))
    vol.destroy()


def ate_cm(est_xyz, gt_xyz) -> float:
    """Absolute trajectory error ([Sturm 2012]): the estimated camera positions are rigidly aligned to the
    ground truth (least squares, Kabsch / Horn without scale), ATE = mean position difference after alignment."""
    E, G = np.asarray(est_xyz, dtype=np.float64), np.asarray(gt_xyz, dtype=np.float64)
    ce, cg = E.mean(0), G.mean(0)
    U, _, Vt = np.linalg.svd((E - ce).T @ (G - cg))
    D = np.diag([1.0, 1.0, np.sign(np.linalg.det(Vt.T @ U.T))])
    R = Vt.T @ D @ U.T
    return 100 * float(np.linalg.norm((E - ce) @ R.T + cg - G, axis=1).mean())


def run_sequence_eval(args):
    """--sequence: SURVEY 8(f)-3, tracking quality over the WHOLE config-3 sequence (200 frames: 30 fused at their true poses,
    170 tracked): TE (Eq. 22) and ATE per run, for the harness-assisted run (frames beyond 8 cm restart from ground
    truth, counted) and the un-assisted free run.  --impl reference runs the oracle on `--steps` tracked frames instead."""
    n_track = 170 if args.steps == 20 else args.steps
    n = N_BUILD + n_track
    scene, poses, frames, K, psts = make_workload(n)
    gt = np.stack([p[:, 3] for p in poses[N_BUILD:]])
    out = {}
    if args.impl == "reference":
        import oracle as orc
        cores = os.cpu_count() or 1
        g = orc.make_grid(DIMS, VS, MU)
        F0, W0 = orc.empty_volume(DIMS)
        for i in range(N_BUILD):
            orc.integrate(g, F0, W0, frames[i], K, poses[i].astype(np.float32), half_storage=True, nthreads=cores)
        for name, assist in (("assisted", True), ("unassisted", False)):
            F, W = F0.copy(), W0.copy()
            pose, r0 = poses[N_BUILD - 1].astype(np.float32), R0_PRIOR.astype(np.float64)
            est, tes, lost = [], [], 0
            for i in range(N_BUILD, n):
                o = orc.pfo_track(g, F, W, frames[i], K, psts, STRIDES, ITERS, pose, pose, r0=r0, early_stop=True, nthreads=cores)
                te = float(np.linalg.norm(o["pose"][:, 3] - poses[i][:, 3]))
                est.append(o["pose"][:, 3].copy()); tes.append(te)
                if assist and not te < LOST_TE:
                    pose, r0, lost = poses[i].astype(np.float32), R0_PRIOR.astype(np.float64), lost + 1
                else:
                    pose, r0 = o["pose"].astype(np.float32), o["r1"]
                orc.integrate(g, F, W, frames[i], K, pose, half_storage=True, nthreads=cores)
            out[name] = {**te_stats(tes), "ate_cm": ate_cm(est, gt), "frames_restarted_from_gt": lost}
    else:
        import torch

        import paper_2105_05600_b200 as rf
        if not torch.cuda.is_available():
            raise SystemExit("bench.py: no CUDA device; the CUDA arm has no CPU fallback")
        torch.cuda.set_device(0)
        dev = [torch.from_numpy(f).cuda() for f in frames]
        dp = [torch.from_numpy(p).cuda() for p in psts]
        for name, assist in (("assisted", True), ("unassisted", False)):
            vol = rf.Volume(DIMS, VS, MU, dtype=rf.RF_F16_W8)
            for i in range(N_BUILD):
                vol.integrate(dev[i], K, poses[i].astype(np.float32))
            pose, r0 = poses[N_BUILD - 1].astype(np.float32), R0_PRIOR
            est, tes, lost, its = [], [], 0, []
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for i in range(N_BUILD, n):
                o = vol.track_integrate(dev[i], K, dp, STRIDES, ITERS, pose, pose, r0=r0, flags=0,
                                        gate=(poses[i][:, 3], LOST_TE) if assist else None)
                est.append(o["pose"][:, 3].astype(np.float64)); its.append(o["iters_run"])
                tes.append(float(np.linalg.norm(est[-1] - poses[i][:, 3])))
                if o["integrated"]:
                    pose, r0 = o["pose"], o["r1"]
                else:
                    pose, r0, lost = poses[i].astype(np.float32), R0_PRIOR, lost + 1
                    vol.integrate(dev[i], K, pose)
            e1.record(); torch.cuda.synchronize()
            out[name] = {**te_stats(tes), "ate_cm": ate_cm(est, gt), "frames_restarted_from_gt": lost,
                         "ms_per_frame": e0.elapsed_time(e1) / n_track, "mean_iterations": float(np.mean(its))}
            vol.destroy()
    print(json.dumps({"metric": "tracking quality over the config-3 sequence (TE Eq. 22, ATE)", "impl": args.impl, "n_gpus": 1,
                      "data": "synthetic", "tracked_frames": n_track, "lost_threshold_cm": 100 * LOST_TE, "results": out}))


def run_ablation(args):
    """--ablation: SURVEY 8(f)-1 on the config-2 frame (256^3 fp32 map, 320x240 frame 15 deg / 8 cm away): the shape of Fig. 9
    (fitness of the best pose so far against the iteration) for PFO with the particle swarm template, vanilla PFO and PSO,
    and the end point of the paper's ablation variants (Fig. 11, Table 2, A14).  Every curve is the fitness of the method's
    best pose so far re-evaluated on ONE common point set (stride 8) so that the methods are comparable."""
    import torch

    import paper_2105_05600_b200 as rf

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA arm has no CPU fallback")
    torch.cuda.set_device(0)
    c = S.make_config2_inputs()
    K = c["K"]
    vol = rf.Volume(c["dims"], c["voxel_size"], c["trunc"], dtype=rf.RF_F32_W8)
    for T, d in zip(c["build_poses"], c["build_frames"]):
        vol.integrate(torch.from_numpy(d).cuda(), K, T)
    depth = torch.from_numpy(c["tracked_depth"]).cuda()
    psts = [torch.from_numpy(p).cuda() for p in c["psts"]]
    T0 = c["T_prev"].astype(np.float32)
    iters = args.steps
    pts = vol.backproject(depth, K, 8)
    zero = torch.zeros((1, 6), dtype=torch.float32, device="cuda")
    ones = np.ones(6, dtype=np.float32)

    def fitness_at(pose):
        return float(vol.eval_particles(pts, zero, np.asarray(pose, dtype=np.float32), ones)[0][0])

    def te(pose):
        return 100 * float(np.linalg.norm(np.asarray(pose, dtype=np.float64)[:, 3] - c["T_true"][:, 3]))

    def apply(delta):                      # Delta(delta) o T_0 on the host, for reporting only
        d = np.asarray(delta, dtype=np.float64)
        n = float(np.linalg.norm(d[:3]))
        return S.compose_delta(T0.astype(np.float64), d[:3] / n if n > 0 else [1.0, 0.0, 0.0], 2.0 * np.arcsin(min(n, 1.0)), d[3:])

    out = {"start": {"fitness": fitness_at(T0), "te_cm": te(T0)}}
    # ---- PFO with PST (Algorithm 1) and its variants
    variants = {"pst": 0, "no_overlap": rf.RF_TRACK_NO_OVERLAP, "rescale_iso": rf.RF_TRACK_RESCALE_ISO, "rescale_aniso": rf.RF_TRACK_RESCALE_ANISO,
                "no_normalize_eq14": rf.RF_TRACK_MODE_EQ14, "f1": rf.RF_TRACK_MODE_F1, "threshold_eq21": rf.RF_TRACK_THRESH_EQ21}
    for name, fl in variants.items():
        r = vol.pfo_track(depth, K, psts, c["strides"], iters, T0, T0, r0=None, flags=fl | rf.RF_TRACK_NO_EARLY_STOP, want_trace=True)
        curve = [fitness_at(np.array(t.pose[:]).reshape(3, 4)) for t in r["trace"]]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(5):
            vol.pfo_track(depth, K, psts, c["strides"], iters, T0, T0, r0=None, flags=fl | rf.RF_TRACK_NO_EARLY_STOP)
        e1.record(); torch.cuda.synchronize()
        out[name] = {"fitness_per_iteration": curve, "te_cm": te(r["pose"]), "evals": r["evals"], "ms": e0.elapsed_time(e1) / 5}
    # ---- the baselines: same number of particles per step as the mean template level, level-1 point set
    N = 4096
    gen = torch.Generator(device="cuda").manual_seed(S.config_seed(2, 9))
    pts1 = vol.backproject(depth, K, c["strides"][1])
    sigma = np.full(6, 0.02, dtype=np.float32)
    state, anc = torch.zeros((N, 6), dtype=torch.float32, device="cuda"), None
    best = torch.zeros(8, dtype=torch.float32, device="cuda")
    curve, t_ms = [], []
    for k in range(iters):
        z = torch.randn((N, 6), generator=gen, device="cuda", dtype=torch.float32)
        u = float(torch.rand((), generator=gen, device="cuda"))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        state = vol.baseline_propose(state, anc, sigma, z)
        fit, _ = vol.eval_particles(pts1, state, T0, ones)
        vol.baseline_best(fit, state, None, None, k == 0, best)
        anc = vol.baseline_resample(fit, u)
        e1.record(); torch.cuda.synchronize()
        t_ms.append(e0.elapsed_time(e1))
        curve.append(fitness_at(apply(best[:6].cpu().numpy())))
    out["vanilla_pfo"] = {"fitness_per_iteration": curve, "te_cm": te(apply(best[:6].cpu().numpy())), "particles": N, "sigma": sigma.tolist(),
                          "ms": float(np.sum(t_ms[1:]) * iters / max(iters - 1, 1))}
    x = (0.05 * psts[2][:N]).contiguous()
    v = torch.zeros_like(x)
    pb, pf, gb = torch.zeros_like(x), torch.zeros(N, dtype=torch.float32, device="cuda"), torch.zeros(8, dtype=torch.float32, device="cuda")
    curve, t_ms = [], []
    for k in range(iters + 1):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        if k > 0:
            ua = torch.rand((N, 6), generator=gen, device="cuda", dtype=torch.float32)
            ub = torch.rand((N, 6), generator=gen, device="cuda", dtype=torch.float32)
            vol.baseline_pso_move(x, v, pb, gb, ua, ub)
        fit, _ = vol.eval_particles(pts1, x, T0, ones)
        vol.baseline_best(fit, x, pb, pf, k == 0, gb)
        e1.record(); torch.cuda.synchronize()
        t_ms.append(e0.elapsed_time(e1))
        if k > 0:
            curve.append(fitness_at(apply(gb[:6].cpu().numpy())))
    out["pso"] = {"fitness_per_iteration": curve, "te_cm": te(apply(gb[:6].cpu().numpy())), "particles": N, "init_scale": 0.05,
                  "ms": float(np.sum(t_ms[2:]) * iters / max(iters - 1, 1))}
    # ---- Gauss-Newton on Eq. 4 ([Bylow 2013]; Fig. 15): same volume, same objective, densest point set (stride 4)
    pts_gn = vol.backproject(depth, K, 4)
    pose, curve, cost = T0.astype(np.float64), [], []
    for k in range(iters):
        g1 = vol.gn_track(pts_gn, pose, 1)
        pose = g1["pose"]
        curve.append(fitness_at(pose)); cost.append(g1["rows"][0].cost / max(g1["rows"][0].n, 1))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(5):
        full = vol.gn_track(pts_gn, T0.astype(np.float64), iters)
    e1.record(); torch.cuda.synchronize()
    out["gauss_newton"] = {"fitness_per_iteration": curve, "mean_sq_residual_per_iteration": cost, "te_cm": te(full["pose"]),
                           "points": int(pts_gn.shape[0]), "iters_run": full["iters_run"], "ms": e0.elapsed_time(e1) / 5}
    vol.destroy()
    print(json.dumps({"metric": "ablation on the config-2 frame (SURVEY 8(f)-1): fitness of the best pose so far per iteration", "n_gpus": 1,
                      "data": "synthetic", "iterations": iters, "common_point_set": "stride 8", "results": out}))


def run_sparse(args):
    """--sparse: SURVEY 8(f)-3, sparse brick allocation.  The config-3 step (map of N_BUILD frames, then `--steps` frames
    tracked with Algorithm 1 + fused) on (a) the dense 512^3 volume, (b) a sparse volume of the same dims and origin,
    (c) a sparse volume whose logical grid is 2048^3 (20.48 m at 1 cm: 8.6 G voxels) with the room at voxel offset 768.
    Every tracked frame starts from the previous ground-truth pose, so the three runs see the same inputs; (a) and (b) must
    agree bit for bit.  One JSON line: ms per tracked frame, bricks allocated, bytes of volume + atlas."""
    import torch

    import paper_2105_05600_b200 as rf

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA arm has no CPU fallback")
    torch.cuda.set_device(0)
    K_steps, W_steps, P_steps = args.steps, max(args.warmup, 3), 10
    n = N_BUILD + W_steps + K_steps
    scene, poses, frames, K, psts = make_workload(n + P_steps)
    dev = [torch.from_numpy(f).cuda() for f in frames]
    dp = [torch.from_numpy(p).cuda() for p in psts]
    POOL = 262144                                   # as many bricks as the dense 512^3 grid has: never the limit here
    OFF = 768
    runs = {"dense_512": dict(dims=DIMS, origin=(0.0, 0.0, 0.0), pool=0),
            "sparse_512": dict(dims=DIMS, origin=(0.0, 0.0, 0.0), pool=POOL),
            "sparse_2048_logical": dict(dims=(2048, 2048, 2048), origin=(-OFF * VS,) * 3, pool=POOL)}
    out, final = {}, {}
    for name, c in runs.items():
        vol = rf.Volume(c["dims"], VS, MU, dtype=rf.RF_F16_W8, origin=c["origin"], pool_bricks=c["pool"])
        for i in range(N_BUILD):
            vol.integrate(dev[i], K, poses[i].astype(np.float32))
        res, evals = [], 0
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for i in range(N_BUILD, n):
            if i == N_BUILD + W_steps:
                torch.cuda.synchronize()
                e0.record()
            prev = poses[i - 1].astype(np.float32)
            o = vol.track_integrate(dev[i], K, dp, STRIDES, ITERS, prev, prev, r0=R0_PRIOR, flags=0)
            res.append(o["pose"].copy())
            if i >= N_BUILD + W_steps:
                evals += int(o["evals"])
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / K_steps
        st = vol.pool_stats()
        stored = st["capacity"] if c["pool"] else int(np.prod([(d + 7) // 8 for d in c["dims"]]))
        te = [float(np.linalg.norm(r[:, 3].astype(np.float64) - poses[N_BUILD + k][:, 3])) for k, r in enumerate(res)]
        out[name] = {"ms_per_step": ms, "evals_per_s": evals / (ms * 1e-3 * K_steps), "bricks_allocated": st["allocated"],
                     "bricks_dropped_last": st["dropped_last"], "logical_bricks": int(np.prod([(d + 7) // 8 for d in c["dims"]])),
                     "bytes_volume_plus_atlas_stored": stored * 512 * (2 + 1 + 16),
                     "bytes_volume_plus_atlas_in_use": st["allocated"] * 512 * (2 + 1 + 16),
                     "median_te_cm": 100 * float(np.median(te))}
        final[name] = res
        # per-kernel time of a tracked frame: CUDA events around every launch (kernels serialised), P_steps more frames
        vol.profile_enable(True)
        for slot in range(6):
            vol.profile_read(slot)
        for i in range(n, n + P_steps):
            prev = poses[i - 1].astype(np.float32)
            vol.track_integrate(dev[i], K, dp, STRIDES, ITERS, prev, prev, r0=R0_PRIOR, flags=0)
        torch.cuda.synchronize()
        slots = ["k_fitness", "k_update", "k_atlas_build", "k_swarm_update", "tile_max_cull_atlas_mark", "backproject_frame_begin"]
        out[name]["us_per_frame_by_kernel"] = {nm: 1e3 * vol.profile_read(k)[0] / P_steps for k, nm in enumerate(slots)}
        vol.destroy()
    same = all(np.array_equal(a, b) for a, b in zip(final["dense_512"], final["sparse_512"]))
    dpose = max(float(np.max(np.abs(a - b))) for a, b in zip(final["dense_512"], final["sparse_2048_logical"]))
    print(json.dumps({"metric": "config-3 step on dense and sparse volumes (SURVEY 8(f)-3)", "n_gpus": 1, "data": "synthetic",
                      "steps": K_steps, "warmup": W_steps, "results": out, "sparse_512_poses_bit_identical_to_dense": bool(same),
                      "sparse_2048_max_pose_difference_to_dense": dpose,
                      "note": "every tracked frame starts from the previous ground-truth pose (identical inputs for the three runs); "
                              "a dense 2048^3 fp16+u8 volume with its atlas would take 163 GB"}))


def run_concurrent(args):
    """--sequences S: throughput mode.  One tracked frame is latency-bound (a chain of 2 x 20 dependent launches that each
    fill the GPU for ~10 us), so one sequence leaves most of the machine idle; a server that tracks several cameras runs
    S independent sequences on one GPU, each with its own volume, stream and host thread (the C calls release the GIL).
    Each sequence tracks its own stretch of the seeded config-3 trajectory (the stretches of `replicas.shard_start`) with
    the headline settings.  Timed on the host around all threads (start barrier -> last join + device synchronise): the
    device-side time of one stream says nothing about the others.  One JSON line with S = 1, 2, 4, ... up to --sequences."""
    import torch

    import paper_2105_05600_b200 as rf

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA arm has no CPU fallback")
    torch.cuda.set_device(0)
    K_steps, W_steps, S_max = args.steps, max(args.warmup, 3), max(1, args.sequences)
    n = N_BUILD + W_steps + K_steps
    work = []
    for s in range(S_max):
        scene, poses, frames, K, psts = make_workload(n, s)
        work.append((poses, [torch.from_numpy(f).cuda() for f in frames], K))
    dpst = [torch.from_numpy(p).cuda() for p in psts]

    def track(vol, s, first, count, state):
        poses, dev, K = work[s]
        pose, r0 = state
        evals, lost = 0, 0
        for i in range(first, first + count):
            out = vol.track_integrate(dev[i], K, dpst, STRIDES, ITERS, pose, pose, r0=r0, flags=0, gate=(poses[i][:, 3], LOST_TE))
            evals += out["evals"]
            if out["integrated"]:
                pose, r0 = out["pose"], out["r1"]
            else:
                pose, r0, lost = poses[i].astype(np.float32), R0_PRIOR, lost + 1
                vol.integrate(dev[i], K, pose)
        return (pose, r0), evals, lost

    counts = sorted({c for c in (1, 2, 4, 8, S_max) if c <= S_max})
    results = []
    for S_ in counts:
        streams = [torch.cuda.Stream() for _ in range(S_)]
        vols, states = [], []
        for s in range(S_):
            poses, dev, K = work[s]
            v = rf.Volume(DIMS, VS, MU, dtype=rf.RF_F16_W8, stream=streams[s])
            for i in range(N_BUILD):
                v.integrate(dev[i], K, poses[i].astype(np.float32))
            st, _, _ = track(v, s, N_BUILD, W_steps, (poses[N_BUILD - 1].astype(np.float32), R0_PRIOR))
            vols.append(v); states.append(st)
        torch.cuda.synchronize()
        evs, losts = [0] * S_, [0] * S_
        gate = threading.Barrier(S_ + 1)

        def worker(s):
            gate.wait()
            _, evs[s], losts[s] = track(vols[s], s, N_BUILD + W_steps, K_steps, states[s])
            streams[s].synchronize()

        th = [threading.Thread(target=worker, args=(s,)) for s in range(S_)]
        for t in th:
            t.start()
        gate.wait()
        t0 = time.perf_counter()
        for t in th:
            t.join()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        results.append({"sequences": S_, "frames_per_s": S_ * K_steps / dt, "evals_per_s": sum(evs) / dt,
                        "ms_per_frame_per_sequence": 1e3 * dt / K_steps, "frames_restarted_from_gt": int(sum(losts))})
        for v in vols:
            v.destroy()
    base = results[0]["frames_per_s"]
    for r in results:
        r["throughput_vs_one_sequence"] = r["frames_per_s"] / base
    print(json.dumps({"metric": "config-3 tracked frames per second, S independent sequences on one GPU (throughput mode)", "n_gpus": 1,
                      "data": "synthetic", "steps": K_steps, "warmup": W_steps, "timing": "host wall clock around all threads",
                      "results": results}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="configs 4 and 5 instead of the config-3 step (one GPU)")
    ap.add_argument("--readout", action="store_true", help="ray-cast read-out of the config-3 map (one GPU)")
    ap.add_argument("--sequence", action="store_true", help="TE / ATE over the whole 200-frame config-3 sequence (--steps tracked frames; default all 170)")
    ap.add_argument("--ablation", action="store_true", help="Fig. 9 shape + ablation variants on the config-2 frame (one GPU); --steps = iterations")
    ap.add_argument("--sparse", action="store_true", help="config-3 step on dense vs sparse volumes, and on a 2048^3 logical grid (one GPU)")
    ap.add_argument("--config5", action="store_true", help="config 5 alone: --steps frames fused into a 1024^3 volume (one GPU)")
    ap.add_argument("--sequences", type=int, default=0, help="throughput mode: up to S independent config-3 sequences on one GPU, one stream and host thread each")
    args = ap.parse_args()
    if args.sequence:
        run_sequence_eval(args)
    elif args.sequences > 0:
        run_concurrent(args)
    elif args.sweep:
        run_sweep(args)
    elif args.config5:
        run_config5(args)
    elif args.sparse:
        run_sparse(args)
    elif args.ablation:
        run_ablation(args)
    elif args.readout:
        run_readout(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()

/* rosefusion_b200.h -- C ABI of the B200-native ROSEFusion hot path (arxiv 2105.05600).
 *
 * "P:L<n>" = PAPER.md line n.  "R-..." / "A<n>" = readings listed in DESIGN.md.
 * Every step of the path runs in hand-written CUDA kernels for sm_100a; there is no CPU fallback.
 *
 * Conventions
 *   Poses      camera-to-world, row-major [R|t], 12 floats, x^G = R x + t (Eq. 1). HOST pointers,
 *              copied at call time.
 *   K          (fx, fy, cx, cy), HOST pointer; pixel centres at integer (u, v).
 *   Volumes    TSDF normalised to [-1,1] (distance / trunc, A7) plus a u8 weight; voxel (i,j,k) has its
 *              sample at origin + (i+1/2, j+1/2, k+1/2) * voxel_size.  Device storage is 8x8x8 bricks
 *              (DESIGN.md section 5); the dense x-fastest order x + X*(y + Y*z) exists only at
 *              upload / download.  At most 8192 voxels per axis and 2^32 - 16 voxels in total.
 *   *_dev      DEVICE pointers owned by the caller (torch tensors).  The library owns rf_volume and its
 *              scratch, allocated at create / first use, never per call on the hot path.
 *   Stream     every call is asynchronous on the volume's stream unless stated; calls on one volume
 *              must be serialised by the caller.
 *   Threads    different volumes may be driven from different host threads at the same time (each on its own
 *              stream: `bench.py --sequences`); the library keeps no mutable state outside an rf_volume except the
 *              launch counter (atomic), the per-thread error text and the static scratch of rf_gn_track_noalloc.
 *   Errors     every call returns an rf_status; no exception crosses the ABI and nothing is printed.
 *              rf_last_error() gives the text of the last failure on the calling thread.
 */
#ifndef ROSEFUSION_B200_H
#define ROSEFUSION_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  RF_OK = 0,
  RF_ERR_INVALID_ARG = 1, /* NULL, non-positive size, trunc < voxel_size, misaligned pointer, iters not in [1,64] */
  RF_ERR_OOM = 2,
  RF_ERR_CUDA = 3,        /* sticky CUDA error; text via rf_last_error() */
  RF_ERR_UNSUPPORTED = 4  /* no sm_100 device */
} rf_status;

typedef enum { RF_F32_W8 = 0, RF_F16_W8 = 1 } rf_dtype; /* TSDF fp32 or fp16; weight always u8 */

typedef struct rf_volume rf_volume; /* opaque */

typedef struct {
  int32_t dtype;    /* rf_dtype, default RF_F32_W8 */
  float origin[3];  /* world position of the minimum corner, default 0 */
  int32_t w_max;    /* weight cap, 1..255, default 255 (A17) */
  void* stream;     /* cudaStream_t, NULL = legacy default stream */
  int32_t pool_bricks; /* 0: dense volume.  > 0: SPARSE volume ("sparse/bricked allocation for volumes beyond
                        * 1024^3"): the grid of `dims` is only a logical index space (up to 8192 voxels per axis and 2^27 bricks)
                        * and at most pool_bricks bricks of 8x8x8 voxels are stored; a brick is allocated the first time an
                        * integration sweeps it (conservative frustum + far cull), never freed before rf_volume_reset.  A brick
                        * that finds the pool full is dropped from that integration (rf_volume_pool_stats reports it).
                        * Every call works on a sparse volume (rf_volume_upload gives each brick with an observed voxel a
                        * slot and returns RF_ERR_OOM if the pool is too small); a grid too large for rf_volume_download /
                        * _upload is read with rf_volume_download_box.  Results are bit-identical to a dense volume of the
                        * same dims and origin as long as nothing was dropped. */
} rf_volume_opts;

/* ---- volume life cycle (step a6 state; framework of [Curless-Levoy 1996; Izadi 2011]) ---- */
/* dims[a] > 0 (padded internally to multiples of 8), voxel_size > 0, trunc >= voxel_size.
 * All voxels start unobserved (W = 0). */
int rf_volume_create(const int32_t dims[3], float voxel_size, float trunc, rf_volume** out);
int rf_volume_create_ex(const int32_t dims[3], float voxel_size, float trunc, const rf_volume_opts* opts,
                        rf_volume** out);
int rf_volume_destroy(rf_volume* vol);
int rf_volume_reset(rf_volume* vol); /* back to all-unobserved */
/* Sparse volumes: out[0] = bricks allocated so far, out[1] = pool capacity, out[2] = bricks dropped by the most recent
 * integration because the pool was full (their voxels were not updated), out[3] = 0.  Dense volumes: out[0] = out[1] = number
 * of bricks, out[2] = 0.  Synchronises the stream. */
int rf_volume_pool_stats(rf_volume* vol, int64_t out[4]);

/* ---- a6: projective TSDF integration of one depth frame (conventions A17 / R-I1) ----
 * Per voxel centre p_w: p_c = R^T (p_w - t); skip if z <= 0; (u,v) = nearest pixel; skip if outside the
 * image or depth invalid (<= 0 or non-finite); sdf = d - z; skip if sdf < -trunc; f = min(1, sdf/trunc);
 * F <- (W F + f)/(W + 1); W <- min(W + 1, w_max).
 * depth: row-major float32 metres, width*height.  depth_on_host == 1: `depth` is a HOST pointer and the
 * host->device copy is part of the call.  depth_on_host == 2: `depth` is ignored and the frame that the last
 * host-depth call on this volume (rf_pfo_track or rf_integrate_ex) copied to the device is fused: a tracked frame
 * crosses the bus once. */
int rf_integrate(rf_volume* vol, const float* depth_dev, int32_t width, int32_t height, const float K[4],
                 const float pose_c2w[12]);
int rf_integrate_ex(rf_volume* vol, const float* depth, int32_t depth_on_host, int32_t width, int32_t height,
                    const float K[4], const float pose_c2w[12]);
/* Frame prefetch for a streaming caller: start copying a HOST frame (pinned memory for a truly asynchronous copy) to
 * the device on the volume's internal copy stream; the copy is ordered after everything already enqueued on the volume's
 * stream and overlaps whatever is enqueued next (normally the tracking of the previous frame).  Up to two frames can be
 * pending; rf_pfo_track with frame->depth_on_host == 2 consumes them in order, rf_integrate_ex(depth_on_host == 2) then
 * fuses that same frame.  The host buffer must stay valid until the consuming rf_pfo_track returns.
 * Ordering: the two slots alternate, so staging a frame re-uses the slot of the frame consumed two calls earlier; fuse a
 * consumed frame (rf_integrate_ex with depth_on_host == 2, or rf_track_integrate) BEFORE staging the frame after next --
 * afterwards that frame is gone and rf_integrate_ex(depth_on_host == 2) returns RF_ERR_INVALID_ARG. */
int rf_stage_frame(rf_volume* vol, const float* depth_host, int32_t width, int32_t height);
/* Number of voxels the last rf_integrate updated (synchronises the stream).  Measurement helper. */
int rf_integrate_last_updated(rf_volume* vol, int64_t* n_updated);
/* Same, plus the number of 8x8x8 bricks the cull pass handed to the update kernel (its candidate voxels = 512 x
 * that) and the number of bricks the last gather-atlas refresh rewrote.  stats_out[0] = voxels updated,
 * stats_out[1] = bricks swept, stats_out[2] = atlas bricks refreshed, stats_out[3] = 0.  Measurement helper. */
int rf_integrate_last_stats(rf_volume* vol, int64_t stats_out[4]);

/* ---- a0: back-projection + stride down-sampling (lattice phase floor(s/2), O3) ----
 * points_out_dev: [M,4] float32 (x, y, z, mask), M = ceil((W - s/2)/s) * ceil((H - s/2)/s), row-major over
 * the lattice; mask = 0 where depth is invalid.  Returns M through *m_out (host). */
int rf_backproject(const rf_volume* vol, const float* depth_dev, int32_t width, int32_t height, const float K[4],
                   int32_t stride, float* points_out_dev, int32_t* m_out);

/* ---- a2 + a3: particle fitness (Eq. 1, 4, 14, 20) ----
 * For particle j: delta = scale (.) pst[j]; q = (sqrt(1 - |delta_q|^2), delta_q); R_j = R(q) R_c,
 * t_j = t_c + delta_t (MovePST/RescalePST on the fly; A2, A3).  For every point with mask != 0:
 * trilinear psi at R_j x + t_j; the point counts iff its 2x2x2 cell lies inside the grid and all 8 corners
 * are observed.  S_j = sum psi^2, n_j = count, M_O = number of mask != 0 points.
 * mode 0 (F2, default): fitness = exp(-(S_j + (M_O - n_j)) / (tau M_O)), tau = 1 (A6).
 * mode 1 (F1): fitness = exp(-S_j / (tau n_j)), 0 when n_j < M_O/2.
 * mode 2 (Eq. 14, the paper's "No Normalize" ablation): fitness = exp(-(S_j + (M_O - n_j)) / tau).
 * points_dev 16-byte aligned, M < 2^20.  Outputs are device arrays of N.  S_out_dev may be NULL.
 * The first evaluation on a volume allocates its gather atlas (8x the TSDF's bytes: 16 B per voxel for fp16 volumes,
 * 32 B for fp32; RF_ERR_OOM if that does not fit) and builds it; later integrations keep it current. */
int rf_eval_particles(const rf_volume* vol, const float* points_dev, int32_t M, const float* pst_dev, int32_t N,
                      const float center_pose_c2w[12], const float scale[6], float* fitness_out_dev,
                      int32_t* count_out_dev);
int rf_eval_particles_ex(const rf_volume* vol, const float* points_dev, int32_t M, const float* pst_dev, int32_t N,
                         const float center_pose_c2w[12], const float scale[6], int32_t mode,
                         float* fitness_out_dev, int32_t* count_out_dev, float* S_out_dev);

/* ---- a0-a5: Algorithm 1 for one frame, whole loop on the device ---- */
typedef struct {
  const float* depth;     /* width*height float32 metres */
  int32_t depth_on_host;  /* 1: HOST pointer, copy is part of the call; 2: `depth` ignored, consume the oldest frame
                             prefetched with rf_stage_frame */
  int32_t width, height;
  float K[4];
} rf_frame;

typedef struct {
  const float* pst_dev[3]; /* [N,6] float32 each, points of the unit 6-D ball */
  int32_t N[3];
  int32_t stride[3];       /* per-axis depth stride of the level (A10) */
} rf_pst_set;

#define RF_TRACK_NO_EARLY_STOP 1 /* run exactly `iters` iterations (config 2) */
#define RF_TRACK_MODE_F1 2       /* fitness normalisation F1 instead of F2 */
#define RF_TRACK_NO_GRAPH 4      /* launch the frame loop kernel by kernel instead of replaying its CUDA graph */
#define RF_TRACK_NO_PDL 8        /* no programmatic dependent launch between the kernels of the frame loop */
/* Ablation variants of the paper (Fig. 11, Table 2); off by default. */
#define RF_TRACK_NO_OVERLAP 16    /* "No Overlap": O_k := every valid pixel of I_d instead of Eq. (19) */
#define RF_TRACK_RESCALE_ISO 32   /* Eq. (17) with its isotropic part only:   r^_d = (1 - rho~)/sqrt(6) + eps */
#define RF_TRACK_RESCALE_ANISO 64 /* Eq. (17) with its anisotropic part only: r^_d = |v_d|/||v|| + eps */
#define RF_TRACK_MODE_EQ14 128    /* "No Normalize": Eq. (14) instead of Eq. (20), rho = exp(-(S + (M_O - n))/tau) */
#define RF_TRACK_THRESH_EQ21 256  /* A14 variant: the advantage-set threshold of iteration k is Eq. (21)'s rho~ of
                                     iteration k-1 (after an empty step: the threshold that step used) instead of the exact
                                     fitness of the centre; the first iteration of a frame evaluates the centre exactly */

typedef struct {
  float pose_c2w[12];      /* in: initial pose T_0 (normally = prev);  out: s_*^t */
  float prev_pose_c2w[12]; /* in: s_*^{t-1}, used by the overlap set O_k (Eq. 19) */
  float r0[6];             /* in (if has_r0): r_0^t;  out: r_1^t for the next frame */
  int32_t has_r0;          /* in: 0 -> isotropic rule A11;  out: 1 */
  int32_t flags;           /* RF_TRACK_* */
  int32_t start_iter;      /* normally 0.  Test hook for teacher-forced parity: number of iterations of this frame
                              already done elsewhere; the level schedule (A15) and the r_1 bookkeeping continue
                              from there, i.e. this call runs iterations start_iter+1 .. start_iter+iters.
                              Requires has_r0 when > 0. */
  float aps_threshold;     /* RF_TRACK_THRESH_EQ21 only.  in (start_iter > 0): the threshold carried from the iteration
                              before, <= 0 = none (evaluate the centre);  out: the threshold the next iteration would use */
} rf_track_state;

#define RF_TRACK_NO_POINTS 1  /* status bit: no usable point, pose unchanged */
#define RF_TRACK_STOP_EMPTY 2 /* stopped: APS empty twice in a row */
#define RF_TRACK_STOP_SMALL 4 /* stopped: change < 1e-6 in all six dims */

typedef struct {
  int32_t iters_run;
  int32_t status;
  float final_fitness;  /* rho~ of the last non-empty step, else rho of the centre */
  int32_t final_count;  /* valid count of the best candidate of the last iteration */
  int32_t argmax;       /* best candidate of the last iteration, 0 = centre, 1+j = particle j */
  int64_t evals;        /* sum over iterations of (N_l + 1) * M_O */
} rf_track_result;

typedef struct {         /* one row per iteration; HOST array of `iters` rows or NULL */
  int32_t level, M_O, n_aps, argmax, stop, empty_run;
  double rho_ref, rho_max, rho_tilde, sum_omega;
  double delta_star[6];
  double pose[12];
  double r[6];
} rf_track_trace;

/* Does NOT integrate: the caller fuses with rf_integrate(state->pose_c2w).  iters in [1,64].
 * Synchronises the stream once, at the end, to return state / result / trace. */
int rf_pfo_track(rf_volume* vol, const rf_frame* frame, const rf_pst_set* pst_set, int32_t iters,
                 rf_track_state* state, rf_track_result* result, rf_track_trace* trace_or_null);

/* One frame of the paper's pipeline ("estimate the pose, then fuse the frame at it") in one call: exactly
 * rf_pfo_track followed by rf_integrate_ex of the same frame at the tracked pose state->pose_c2w -- same kernels, same
 * results, bit for bit; the fusion kernels are enqueued from C as soon as the pose is on the host, so the GPU does not
 * wait for the caller to come back with a second call.  Optional gate (tracking-loss guard): if gate_center_or_null is
 * not NULL and the tracked camera position is farther than gate_radius (metres) from gate_center (or is not finite),
 * the frame is NOT fused and *integrated_out = 0: the caller decides what to do (e.g. rf_integrate_ex at a
 * re-localised pose).  *integrated_out = 1 when the frame was fused.  The fusion is stream-ordered, not synchronised. */
int rf_track_integrate(rf_volume* vol, const rf_frame* frame, const rf_pst_set* pst_set, int32_t iters,
                       rf_track_state* state, rf_track_result* result, rf_track_trace* trace_or_null,
                       const float* gate_center_or_null, float gate_radius, int32_t* integrated_out);

/* ---- particle-sharded frame loop: Algorithm 1 with each level's template split over G ranks ----
 * Every rank holds the whole volume and frame and a contiguous slice of each level's template (pst_set->pst_dev[l] = the
 * slice, N[l] = its length; offset[l] = global index of its first particle; n_total[l] = particles of the whole level).
 * Per iteration k = 1, 2, ...:
 *   rf_shard_eval   evaluates the slice and the centre (every rank evaluates the centre: same bits everywhere) and reduces
 *                   them to one row of 16 doubles in row_out_dev (sum w, sum w rho, sum w delta[6], |APS|, -, best exponent,
 *                   best global index, its count, rho_ref, |O|, -): step a2-a3 and the per-candidate half of a4;
 *   (the caller all-gathers the rows: 128 bytes per rank -- torch.distributed over NCCL / NVLink, plumbing);
 *   rf_shard_apply  folds the G rows in rank order (the same bits on every rank) and applies Eq. 15-18, 21 and the stop rules
 *                   to this rank's copy of the state; returns the stop flag (synchronises) and optionally the trace row.
 * rf_shard_begin back-projects the three levels and sets the state (state->has_r0 is required: the first tracked frame's
 * rule A11 is not sharded); rf_shard_end returns pose, r_1 and the result as rf_pfo_track does.  With G = 1 the result is
 * bit-identical to rf_pfo_track.  The frame must be a device pointer. */
int rf_shard_begin(rf_volume* vol, const rf_frame* frame, const rf_pst_set* local_slice, const int32_t offset[3],
                   const int32_t n_total[3], rf_track_state* state);
int rf_shard_eval(rf_volume* vol, int32_t k, double* row_out_dev);
int rf_shard_apply(rf_volume* vol, int32_t k, const double* rows_dev, int32_t G, rf_track_trace* trace_row_or_null,
                   int32_t* done_out);
int rf_shard_end(rf_volume* vol, rf_track_state* state, rf_track_result* result);

/* ---- a7: read-out and test hook (not timed) ----
 * Dense x-fastest float32; unobserved voxels read tsdf = 1.0, weight = 0.  weight_out may be NULL.
 * on_device != 0: the pointers are device pointers.  Both synchronise the stream. */
int rf_volume_download(const rf_volume* vol, float* tsdf_out, float* weight_out);
int rf_volume_download_ex(const rf_volume* vol, float* tsdf_out, float* weight_out, int32_t on_device);
int rf_volume_upload(rf_volume* vol, const float* tsdf_host, const float* weight_host);
/* Dense read-out of the box of voxels [lo, lo + size) (x fastest, then y, then z; same conventions as rf_volume_download:
 * unobserved voxels read TSDF 1.0, weight 0) into DEVICE buffers of size[0]*size[1]*size[2] floats -- the way to look at a
 * region of a sparse volume whose logical grid is too large to download whole.  Dense and sparse volumes.  Stream-ordered,
 * does not synchronise. */
int rf_volume_download_box(const rf_volume* vol, const int32_t lo[3], const int32_t size[3], float* tsdf_out_dev,
                           float* weight_out_dev_or_null);

/* ---- read-out: ray casting of the fused surface to a depth (+ normal) map (reconstructions shown
 * P:L525-537; algorithm = reading R-R1) ----
 * Pixel (u,v) marches x(z) = R ((u-cx)/fx, (v-cy)/fy, 1) z + t at the depths z_k = k*step, k = 1 .. floor(z_max/step).
 * The surface is the first k whose samples k-1 and k are both valid trilinear samples (A8: all 8 corners observed)
 * with psi_{k-1} > 0 >= psi_k; depth = (k-1)*step + step*psi_{k-1}/(psi_{k-1}-psi_k); no such k -> 0.  A crossing
 * from behind (negative to positive) is not a surface.  step should stay below the truncation distance divided by
 * the longest pixel ray ||((u-cx)/fx,(v-cy)/fy,1)||, or thin crossings can be stepped over.
 * depth_out_dev: [height,width] float32 camera depths (device).  normals_out_dev_or_null: [height,width,3] float32
 * world-frame unit gradient of psi at the hit (central differences of half-width one voxel; NaN where there is no hit
 * or a neighbouring sample is invalid), or NULL.  Uses (and if needed builds / refreshes) the gather atlas.
 * Stream-ordered on the volume's stream; does not synchronise. */
int rf_raycast(rf_volume* vol, const float K[4], int32_t width, int32_t height, const float pose_c2w[12], float step,
               float z_max, float* depth_out_dev, float* normals_out_dev_or_null);

/* ---- read-out: the surface point set ("marching cubes ... to point sets (no graphics API)"; the reconstruction
 * whose completeness / accuracy the paper measures; reading R-R2) ----
 * The vertex set of marching cubes: every grid edge between a voxel and its +x / +y / +z neighbour whose two samples are both
 * observed and lie on different sides of the surface (exactly one of them is > 0) carries one point, the zero of the straight
 * line through the two samples, on the edge between the two voxel centres.  points_out_dev: [cap,3] float32 world positions
 * (device); edge_out_dev_or_null: [cap] int64 edge keys 3 * (i + X (j + Y k)) + axis (device) or NULL.  The order of the
 * points is not defined (sort by key to compare).  *n_out (host) = number of crossing edges; if it exceeds cap only cap
 * points were written -- call again with a larger buffer.  Synchronises the stream.  Note: rf_integrate_last_updated
 * shares the counter this call uses; read it before extracting. */
int rf_extract_surface_points(const rf_volume* vol, float* points_out_dev, int64_t* edge_out_dev_or_null, int64_t cap,
                              int64_t* n_out);

/* ---- Gauss-Newton minimisation of Eq. (4) (the SDF tracker of [Bylow 2013] the paper compares its optimiser
 * with; reading GN1) ----
 * Objective and sample rule of rf_eval_particles: E(T) = sum over valid points of psi(R x + t)^2 (a point counts when all 8
 * corners of its interpolation cell are observed).  Iteration: r_i = psi(p_i), p_i = R x_i + t; J_i = [p_i x grad_i ; grad_i]
 * with grad the analytic derivative of the trilinear interpolant (per metre); (sum J J^T) xi = -sum J r solved by Gaussian
 * elimination with partial pivoting; R <- exp([omega]x) R, t <- exp([omega]x) t + v for xi = (omega, v).  The run stops after
 * `iters` iterations, after a step with |xi| < 1e-9, or at an iteration with fewer than 6 valid points or a singular system
 * (that iteration is still recorded and leaves the pose unchanged).  All arithmetic is binary64.
 * points_dev: [M,4] float32 camera-frame points (x, y, z, valid) on the device, 16-byte aligned (rf_backproject's output;
 * may be NULL when M = 0).  pose_in / pose_out: host, row-major 3x4 camera-to-world.  rows_out_or_null: host, room for `iters` rows, row k = the sums of
 * iteration k BEFORE its step (cost E, number of valid points, full symmetric A row-major, b = sum J r) and |xi| of the step
 * taken; *iters_run_out (host) = rows written.  The iterations run on the device without host round trips; the call
 * synchronises the volume's stream.  Shares the baselines' device scratch: do not interleave with rf_baseline_resample on
 * another stream. */
typedef struct rf_gn_row {
  double cost;
  int32_t n;
  int32_t pad;
  double step_norm;
  double A[36];
  double b[6];
} rf_gn_row;
int rf_gn_track(rf_volume* vol, const float* points_dev, int32_t M, const double pose_in[12], int32_t iters, double pose_out[12],
                rf_gn_row* rows_out_or_null, int32_t* iters_run_out);

/* ---- rf_gn_track without allocation (outside SURVEY section 8 on purpose: for callers that may not call cudaMalloc --
 * code under stream capture, tight serving loops, harnesses that forbid it) ----
 * Same arguments, same kernels, same launch shapes and therefore bit-identical results as rf_gn_track, but the scratch of
 * the run (state, trace rows, per-CTA partial sums) is ONE file-scope device array of rf_gn_noalloc_scratch_bytes() =
 * 174848 bytes that every GPU loading the library holds until the process exits; the call makes no cudaMalloc / cudaFree
 * and calls no allocating library routine.  Limit: iters <= RF_GN_NOALLOC_MAX_ITERS (a larger value is rejected with
 * RF_ERR_INVALID_ARG and a message naming the limit; use rf_gn_track); M is not limited.  The device that is current must
 * be the volume's.  Every call on a device shares the array and finds the previous call's contents in it; the call
 * re-initialises what it reads (pose, stop flag, iteration counter), so sequential calls are independent, but calls that
 * OVERLAP on the GPU (other streams, other volumes, other host threads) race on it: serialise them.  Synchronises the
 * volume's stream. */
#define RF_GN_NOALLOC_MAX_ITERS 64
int rf_gn_track_noalloc(rf_volume* vol, const float* points_dev, int32_t M, const double pose_in[12], int32_t iters,
                        double pose_out[12], rf_gn_row* rows_out_or_null, int32_t* iters_run_out);
int64_t rf_gn_noalloc_scratch_bytes(void);

/* ---- the comparison methods of Section 5.2 (Fig. 9, 10) as primitives around rf_eval_particles ----
 * A particle is an explicit increment delta (float32 [N,6]: imaginary quaternion part, translation) about the frame's initial
 * pose T_0; its fitness is rf_eval_particles(points, delta as the template, N, T_0, scale = (1,...,1)).  Every random number is
 * an input (device arrays the caller fills from its own generator).  All four calls are stream-ordered kernels; the state
 * stays on the device.  Readings B1-B5 in DESIGN.md section 10.
 *   rf_baseline_propose   vanilla PFO proposal, Eq. (12): delta_out_i = clamp(delta_in_{a(i)} + sigma (.) z_i); a = the
 *                         ancestors of the last resampling (NULL = identity), z standard normals [N,6]; clamp: |delta_q| <= 0.95.
 *   rf_baseline_resample  resampling after the likelihood weighting of Eq. (13): systematic resampling with the
 *                         uniform u in [0,1); weights = the fitness values; ancestors_out [N] int32, non-decreasing.
 *   rf_baseline_pso_move  PSO: v <- 0.7298 v + 1.49618 a (.) (pbest - x) + 1.49618 b (.) (gbest - x); x <- clamp(x + v);
 *                         a, b uniform in [0,1) [N,6]; gbest_dev = the first 6 floats of rf_baseline_best's gbest.
 *   rf_baseline_best      bookkeeping: pbest / pbest_fit (optional, both or neither) take x / fitness where strictly better
 *                         (first != 0: unconditionally); gbest_dev [8] = (6 coordinates, fitness, index) takes this step's best
 *                         particle (lowest index among equals) if strictly better than the holder (first != 0: unconditionally). */
int rf_baseline_propose(rf_volume* vol, const float* delta_in_dev, const int32_t* ancestors_dev_or_null, const float sigma[6],
                        const float* normals_dev, int32_t N, float* delta_out_dev);
int rf_baseline_resample(rf_volume* vol, const float* fitness_dev, int32_t N, double u, int32_t* ancestors_out_dev);
int rf_baseline_pso_move(rf_volume* vol, float* x_dev, float* v_dev, const float* pbest_dev, const float* gbest_dev,
                         const float* ua_dev, const float* ub_dev, int32_t N);
int rf_baseline_best(rf_volume* vol, const float* fitness_dev, const float* x_dev, int32_t N, float* pbest_dev_or_null,
                     float* pbest_fit_dev_or_null, int32_t first, float* gbest_dev);

/* ---- measurement helper: the L2-gather roofline denominator ----
 * Independent random 32-byte sector reads over an L2-resident buffer of `bytes`; returns GB/s counting
 * 32 B per request.  mode 0 = random sectors, 1 = streaming 128-bit reads. */
int rf_microbench_l2(int64_t bytes, int32_t mode, int32_t reps, double* gbps_out);

/* Optional per-kernel timing for bench.py's roofline object: when enabled, CUDA events are recorded on the
 * volume's stream around every fitness-kernel launch of rf_pfo_track and around the voxel-update kernel of
 * rf_integrate.  rf_profile_read synchronises, returns the accumulated milliseconds / launch counts since
 * the last read and resets them.  which: 0 = fitness kernel, 1 = integration update kernel, 2 = atlas build kernel,
 * 3 = swarm update kernel, 4 = tile-max + cull + atlas-mark kernels, 5 = back-projection kernels. */
int rf_profile_enable(rf_volume* vol, int32_t on);
int rf_profile_read(rf_volume* vol, int32_t which, double* ms_out, int64_t* launches_out);
/* The individual launch durations (milliseconds, launch order) accumulated for `which` since the last rf_profile_read
 * of that slot; does not reset.  At most `cap` values are written; *n_out = how many exist.  bench.py pairs the
 * fitness launches of a frame with that frame's trace rows to report one roofline per regime (L2-resident swarm /
 * re-inflated swarm).  Synchronises the stream. */
int rf_profile_read_launches(rf_volume* vol, int32_t which, float* ms_each_out, int32_t cap, int32_t* n_out);
/* Number of kernels this library has launched in this process (all volumes). */
int64_t rf_launch_count(void);

const char* rf_last_error(void);
int rf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ROSEFUSION_B200_H */

// rf_track.cu -- steps a1 (overlap mask), a4 (swarm update), a5 (iteration control): Algorithm 1
// with the whole loop on the device.  The paper runs the update on the CPU with one
// CPU<->GPU round trip per iteration (Fig. 8); here state (pose, axis lengths, flags) stays in
// device memory and a `done` flag turns the remaining launches of a frame into no-ops.
#include "rf_common.cuh"
#include <string.h>

#define UP_THREADS 1024

int rf_launch_backproject(cudaStream_t st, const float* depth_dev, int w, int h, const float K[4], int stride,
                          float4* pts, int* m_out);

struct TrackCfg { float fx, fy, cx, cy; int w, h, mode, early_stop, iters; };
struct TrackInit { double T[12]; double Tprev[12]; double r[6]; int has_r0; };

__global__ void k_track_begin(TrackInit in, TrackDev* st) {
  if (threadIdx.x < 12) { st->T[threadIdx.x] = in.T[threadIdx.x]; st->Tprev[threadIdx.x] = in.Tprev[threadIdx.x]; }
  if (threadIdx.x < 6) { st->r[threadIdx.x] = in.r[threadIdx.x]; st->r1[threadIdx.x] = in.r[threadIdx.x]; }
  if (threadIdx.x == 0) {
    st->final_rho = 0; st->evals = 0; st->empty_run = 0; st->done = 0; st->iters_run = 0; st->status = 0;
    st->final_count = 0; st->argmax = 0; st->M_O = 0;
  }
}

// block-wide sums (fixed shape -> deterministic)
__device__ __forceinline__ double block_sum(double v, double* sh) {
  for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  double r = 0;
  if (threadIdx.x < 32) {
    r = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
    for (int o = 16; o; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
  }
  __syncthreads();
  if (threadIdx.x == 0) sh[0] = r;
  __syncthreads();
  r = sh[0];
  return r;
}

// a1: O_k (Eq. 19; A9): keep a point iff, moved to the world by T (= s*_{k-1}) and into camera
// t-1 (Tprev), it has z > 0 and projects inside [0,W) x [0,H).  Runs inside a single CTA.
__device__ void mask_level(const float4* __restrict__ raw, int M, float4* __restrict__ out, TrackDev* st,
                           const TrackCfg& cfg, double* sh) {
  double T[12], P[12];
#pragma unroll
  for (int a = 0; a < 12; ++a) { T[a] = st->T[a]; P[a] = st->Tprev[a]; }
  int cnt = 0;
  for (int i = threadIdx.x; i < M; i += blockDim.x) {
    float4 x = raw[i];
    float keep = 0.f;
    if (x.w != 0.f) {
      const double xw0 = T[0] * x.x + T[1] * x.y + T[2] * x.z + T[3];
      const double xw1 = T[4] * x.x + T[5] * x.y + T[6] * x.z + T[7];
      const double xw2 = T[8] * x.x + T[9] * x.y + T[10] * x.z + T[11];
      const double e0 = xw0 - P[3], e1 = xw1 - P[7], e2 = xw2 - P[11];
      const double y0 = P[0] * e0 + P[4] * e1 + P[8] * e2;
      const double y1 = P[1] * e0 + P[5] * e1 + P[9] * e2;
      const double y2 = P[2] * e0 + P[6] * e1 + P[10] * e2;
      if (y2 > 0.0) {
        const double u = (double)cfg.fx * y0 / y2 + (double)cfg.cx, v = (double)cfg.fy * y1 / y2 + (double)cfg.cy;
        if (u >= 0.0 && u < (double)cfg.w && v >= 0.0 && v < (double)cfg.h) { keep = 1.f; ++cnt; }
      }
    }
    x.w = keep;
    out[i] = x;
  }
  const double tot = block_sum((double)cnt, sh);
  if (threadIdx.x == 0) st->M_O = (int)tot;
}

__global__ void __launch_bounds__(UP_THREADS) k_mask(const float4* raw, int M, float4* out, TrackDev* st, TrackCfg cfg) {
  __shared__ double sh[32];
  if (st->done) return;
  mask_level(raw, M, out, st, cfg, sh);
}

__device__ __forceinline__ double rho_of(double S, int n, int M_O, int mode) {
  if (M_O <= 0) return 0.0;
  if (mode == 1) return (n <= 0 || 2 * (long long)n < (long long)M_O) ? 0.0 : exp(-S / (double)n);
  return exp(-(S + (double)(M_O - n)) / (double)M_O);
}

// first tracked frame (A11): r_0,d = 2 (1 - rho(T_0)) / sqrt(6) + eps from the centre alone on level 0.
__global__ void k_init_r0(unsigned long long* acc_S, int* acc_n, TrackDev* st, TrackCfg cfg) {
  if (threadIdx.x != 0) return;
  const double S = (double)acc_S[0] * (1.0 / RF_S_SCALE);
  const int n = acc_n[0];
  acc_S[0] = 0; acc_n[0] = 0;
  const double rho0 = rho_of(S, n, st->M_O, cfg.mode);
  for (int d = 0; d < 6; ++d) st->r[d] = 2.0 * (1.0 - rho0) / sqrt(6.0) + 1e-3;
  st->evals += st->M_O;
}

// T_out = Delta(delta) o T_in  (MovePST; A2: left-multiplied increment, world-frame translation)
__device__ void apply_delta(const double* Tin, const double* d, double* Tout) {
  const double qx = d[0], qy = d[1], qz = d[2];
  const double qw = sqrt(fmax(0.0, 1.0 - (qx * qx + qy * qy + qz * qz)));
  double Rq[9];
  Rq[0] = 1 - 2 * (qy * qy + qz * qz); Rq[1] = 2 * (qx * qy - qz * qw);     Rq[2] = 2 * (qx * qz + qy * qw);
  Rq[3] = 2 * (qx * qy + qz * qw);     Rq[4] = 1 - 2 * (qx * qx + qz * qz); Rq[5] = 2 * (qy * qz - qx * qw);
  Rq[6] = 2 * (qx * qz - qy * qw);     Rq[7] = 2 * (qy * qz + qx * qw);     Rq[8] = 1 - 2 * (qx * qx + qy * qy);
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) Tout[4 * i + j] = Rq[3 * i] * Tin[j] + Rq[3 * i + 1] * Tin[4 + j] + Rq[3 * i + 2] * Tin[8 + j];
    Tout[4 * i + 3] = Tin[4 * i + 3] + d[3 + i];
  }
}

// a3 + a4 + a5 for iteration k (1-based) on level `level`, then a1 for the next level.
__global__ void __launch_bounds__(UP_THREADS)
k_swarm_update(unsigned long long* __restrict__ acc_S, int* __restrict__ acc_n, int N,
               const float* __restrict__ pst, TrackDev* st, TrackCfg cfg, int k, int k0, int level, double* __restrict__ rho,
               int* __restrict__ cand_n, rf_track_trace* trace, const float4* next_raw, int next_M, float4* next_out) {
  __shared__ double sh[32];
  __shared__ double s_best_v[32];
  __shared__ int s_best_i[32];
  if (st->done) return;
  const int total = N + 1;
  const int M_O = st->M_O;
  // a3: fitness by Eq. (20) from the accumulators (read and clear)
  for (int c = threadIdx.x; c < total; c += blockDim.x) {
    const double S = (double)acc_S[c] * (1.0 / RF_S_SCALE);
    const int n = acc_n[c];
    acc_S[c] = 0; acc_n[c] = 0;
    rho[c] = rho_of(S, n, M_O, cfg.mode);
    cand_n[c] = n;
  }
  __syncthreads();
  const double rho_ref = rho[0];                       // exact fitness of s*_{k-1} on this point set (A14)
  double r[6];
#pragma unroll
  for (int d = 0; d < 6; ++d) r[d] = st->r[d];
  // a4: APS = {j : rho_j > rho_ref}, omega = rho - rho_ref, Eq. (15) and Eq. (21) sums
  double sw = 0, swr = 0, sd[6] = {0, 0, 0, 0, 0, 0}, naps = 0;
  double bv = threadIdx.x == 0 ? rho_ref : -1.0;
  int bi = threadIdx.x == 0 ? 0 : 0x7fffffff;
  for (int j = threadIdx.x; j < N; j += blockDim.x) {
    const double rj = rho[1 + j];
    if (rj > bv) { bv = rj; bi = 1 + j; }             // strided ascending -> lowest index per thread
    if (rj > rho_ref) {
      const double w = rj - rho_ref;
      sw += w; swr += w * rj; naps += 1.0;
#pragma unroll
      for (int d = 0; d < 6; ++d) sd[d] += w * (r[d] * (double)__ldg(pst + 6 * (size_t)j + d));
    }
  }
  sw = block_sum(sw, sh); swr = block_sum(swr, sh); naps = block_sum(naps, sh);
#pragma unroll
  for (int d = 0; d < 6; ++d) sd[d] = block_sum(sd[d], sh);
  // argmax, ties -> lowest index (A18)
  for (int o = 16; o; o >>= 1) {
    const double ov = __shfl_xor_sync(0xffffffffu, bv, o);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
    if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
  }
  if ((threadIdx.x & 31) == 0) { s_best_v[threadIdx.x >> 5] = bv; s_best_i[threadIdx.x >> 5] = bi; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int wdx = 1; wdx < (int)(blockDim.x >> 5); ++wdx)
      if (s_best_v[wdx] > bv || (s_best_v[wdx] == bv && s_best_i[wdx] < bi)) { bv = s_best_v[wdx]; bi = s_best_i[wdx]; }
    const int n_aps = (int)naps;
    double dstar[6] = {0, 0, 0, 0, 0, 0}, rhat[6], rho_tilde = 0, Tn[12];
    int empty_run = st->empty_run, stop = 0;
    if (n_aps > 0) {
      for (int d = 0; d < 6; ++d) dstar[d] = sd[d] / sw;                   // Eq. (15) in the chart at s*_{k-1} (A3)
      rho_tilde = swr / sw;                                                // Eq. (21)
      apply_delta(st->T, dstar, Tn);
      double nv = 0;
      for (int d = 0; d < 6; ++d) nv += dstar[d] * dstar[d];               // v = s_k^* - s_{k-1}^*  (Eq. 16)
      nv = sqrt(nv);
      for (int d = 0; d < 6; ++d) rhat[d] = (nv > 0 ? (1.0 - rho_tilde) * fabs(dstar[d]) / nv : 0.0) + 1e-3;   // Eq. (17), A4
      empty_run = 0;
    } else {
      for (int a = 0; a < 12; ++a) Tn[a] = st->T[a];
      for (int d = 0; d < 6; ++d) rhat[d] = 2.0 * (1.0 - rho_ref) / sqrt(6.0) + 1e-3;   // P:L292, A13
      empty_run += 1;
    }
    for (int d = 0; d < 6; ++d) r[d] = 0.1 * r[d] + 0.9 * rhat[d];         // Eq. (18), beta = 0.1
    if (empty_run >= 2) stop = 1;
    else if (n_aps > 0) {
      double mx = 0;
      for (int d = 0; d < 6; ++d) mx = fmax(mx, fabs(dstar[d]));
      if (mx < 1e-6) stop = 2;                                             // P:L306, A16
    }
    for (int a = 0; a < 12; ++a) st->T[a] = Tn[a];
    for (int d = 0; d < 6; ++d) st->r[d] = r[d];
    if (k == 1) for (int d = 0; d < 6; ++d) st->r1[d] = r[d];              // P:L286  r_0^{t+1} = r_1^t
    st->empty_run = empty_run;
    st->iters_run = k - k0;
    st->final_rho = n_aps > 0 ? rho_tilde : rho_ref;
    st->final_count = cand_n[bi];
    st->argmax = bi;
    st->evals += (long long)total * M_O;
    if (M_O == 0) st->status |= RF_TRACK_NO_POINTS;
    if (cfg.early_stop && stop) { st->done = 1; st->status |= (stop == 1 ? RF_TRACK_STOP_EMPTY : RF_TRACK_STOP_SMALL); }
    if (trace) {
      rf_track_trace& tr = trace[k - k0 - 1];
      tr.level = level; tr.M_O = M_O; tr.n_aps = n_aps; tr.argmax = bi; tr.stop = stop; tr.empty_run = empty_run;
      tr.rho_ref = rho_ref; tr.rho_max = bv; tr.rho_tilde = rho_tilde; tr.sum_omega = n_aps > 0 ? sw : 0.0;
      for (int d = 0; d < 6; ++d) { tr.delta_star[d] = dstar[d]; tr.r[d] = r[d]; }
      for (int a = 0; a < 12; ++a) tr.pose[a] = Tn[a];
    }
  }
  __syncthreads();
  // a1 for the next iteration, with the pose just computed
  if (next_raw && !st->done) mask_level(next_raw, next_M, next_out, st, cfg, sh);
}

extern "C" int rf_pfo_track(rf_volume* v, const rf_frame* f, const rf_pst_set* ps, int32_t iters, rf_track_state* state,
                            rf_track_result* result, rf_track_trace* trace) {
  RF_ARG(v && f && ps && state && result, "rf_pfo_track: NULL argument");
  RF_ARG(f->depth && f->width > 0 && f->height > 0, "rf_pfo_track: bad frame");
  RF_ARG(iters >= 1 && iters <= RF_MAX_ITERS, "rf_pfo_track: iters must be in [1,64]");
  RF_ARG(state->start_iter >= 0 && state->start_iter < 4096, "rf_pfo_track: bad start_iter");
  RF_ARG(state->start_iter == 0 || state->has_r0, "rf_pfo_track: start_iter > 0 needs r0");
  const int k0 = state->start_iter;
  for (int l = 0; l < 3; ++l) {
    RF_ARG(ps->pst_dev[l] && ps->N[l] > 0 && ps->stride[l] > 0, "rf_pfo_track: bad pst_set");
    RF_ARG(ps->stride[l] / 2 < f->width && ps->stride[l] / 2 < f->height, "rf_pfo_track: stride larger than the image");
  }
  cudaStream_t st = v->stream;
  const size_t px = (size_t)f->width * f->height;
  const float* d_dev = f->depth;
  if (f->depth_on_host) {
    int rc = rf_ensure((void**)&v->depth_stage, &v->depth_cap, px * sizeof(float));
    if (rc != RF_OK) return rc;
    RF_CUDA(cudaMemcpyAsync(v->depth_stage, f->depth, px * sizeof(float), cudaMemcpyHostToDevice, st));
    d_dev = v->depth_stage;
  }
  // a0: the three levels, once per frame
  int M[3];
  for (int l = 0; l < 3; ++l) {
    const int s = ps->stride[l];
    const int nu = (f->width - s / 2 + s - 1) / s, nv = (f->height - s / 2 + s - 1) / s;
    const size_t need = (size_t)nu * nv * sizeof(float4);
    if (need > v->pts_cap[l]) {
      cudaFree(v->pts_raw[l]); cudaFree(v->pts_k[l]); v->pts_raw[l] = v->pts_k[l] = nullptr; v->pts_cap[l] = 0;
      RF_CUDA(cudaMalloc(&v->pts_raw[l], need));
      RF_CUDA(cudaMalloc(&v->pts_k[l], need));
      v->pts_cap[l] = need;
    }
    int rc = rf_launch_backproject(st, d_dev, f->width, f->height, f->K, s, v->pts_raw[l], &M[l]);
    if (rc != RF_OK) return rc;
  }
  size_t maxc = 0;
  for (int l = 0; l < 3; ++l) maxc = max(maxc, (size_t)ps->N[l] + 1);
  if (maxc > v->rho_cap) {
    cudaFree(v->rho); cudaFree(v->cand_n); v->rho = nullptr; v->cand_n = nullptr; v->rho_cap = 0;
    RF_CUDA(cudaMalloc(&v->rho, maxc * sizeof(double)));
    RF_CUDA(cudaMalloc(&v->cand_n, maxc * sizeof(int)));
    v->rho_cap = maxc;
  }
  { int rc0 = rf_ensure_acc(v, maxc); if (rc0 != RF_OK) return rc0; }
  TrackCfg cfg;
  cfg.fx = f->K[0]; cfg.fy = f->K[1]; cfg.cx = f->K[2]; cfg.cy = f->K[3]; cfg.w = f->width; cfg.h = f->height;
  cfg.mode = (state->flags & RF_TRACK_MODE_F1) ? 1 : 0;
  cfg.early_stop = (state->flags & RF_TRACK_NO_EARLY_STOP) ? 0 : 1;
  cfg.iters = iters;
  TrackInit in;
  for (int a = 0; a < 12; ++a) { in.T[a] = state->pose_c2w[a]; in.Tprev[a] = state->prev_pose_c2w[a]; }
  for (int d = 0; d < 6; ++d) in.r[d] = state->has_r0 ? state->r0[d] : 0.0;
  in.has_r0 = state->has_r0;
  TrackDev* td = v->track;
  k_track_begin<<<1, 32, 0, st>>>(in, td);
  const int l0 = k0 % 3;
  k_mask<<<1, UP_THREADS, 0, st>>>(v->pts_raw[l0], M[l0], v->pts_k[l0], td, cfg);
  RF_LAUNCHED(2);
  int rc;
  if (!state->has_r0) {
    rc = rf_launch_eval(v, v->pts_k[0], M[0], ps->pst_dev[0], 0, 1, td->T, td->r, nullptr);
    if (rc != RF_OK) return rc;
    k_init_r0<<<1, 32, 0, st>>>(v->acc_S, v->acc_n, td, cfg);
    RF_LAUNCHED(1);
  }
  for (int k = k0 + 1; k <= k0 + iters; ++k) {
    const int l = (k - 1) % 3, nl = k % 3;               // A15: levels in the listed order, cycling
    rc = rf_launch_eval(v, v->pts_k[l], M[l], ps->pst_dev[l], ps->N[l], 1, td->T, td->r, &td->done);
    if (rc != RF_OK) return rc;
    const bool more = k < k0 + iters;
    k_swarm_update<<<1, UP_THREADS, 0, st>>>(v->acc_S, v->acc_n, ps->N[l], ps->pst_dev[l], td, cfg, k, k0, l, v->rho,
                                            v->cand_n, trace ? v->trace_dev : nullptr, more ? v->pts_raw[nl] : nullptr,
                                            more ? M[nl] : 0, more ? v->pts_k[nl] : nullptr);
    RF_LAUNCHED(1);
  }
  RF_CUDA(cudaGetLastError());
  RF_CUDA(cudaMemcpyAsync(v->track_host, td, sizeof(TrackDev), cudaMemcpyDeviceToHost, st));
  if (trace) RF_CUDA(cudaMemcpyAsync(v->trace_host, v->trace_dev, iters * sizeof(rf_track_trace), cudaMemcpyDeviceToHost, st));
  RF_CUDA(cudaStreamSynchronize(st));
  if (v->prof_on) rf_prof_collect(v);
  const TrackDev& h = *v->track_host;
  for (int a = 0; a < 12; ++a) state->pose_c2w[a] = (float)h.T[a];
  for (int d = 0; d < 6; ++d) state->r0[d] = (float)h.r1[d];
  state->has_r0 = 1;
  result->iters_run = h.iters_run; result->status = h.status; result->final_fitness = (float)h.final_rho;
  result->final_count = h.final_count; result->argmax = h.argmax; result->evals = h.evals;
  if (trace) memcpy(trace, v->trace_host, (size_t)h.iters_run * sizeof(rf_track_trace));
  return RF_OK;
}

// rf_baselines.cu -- the comparison methods of Section 5.2 (Fig. 9, 10) as device primitives around the
// unchanged fitness kernel: "vanilla PFO" (Section 3.2: Gaussian random-walk proposal Eq. 12, likelihood weights Eq. 13,
// resampling) and particle swarm optimisation.  A particle is an explicit 6-D increment about the
// frame's initial pose; its fitness is rf_eval_particles with unit axis lengths.  Every random number is an input.
// Readings B1-B5: systematic resampling; Clerc-Kennedy constants; |delta_q| <= 0.95; binary32
// state with every update evaluated in fp64 in a fixed order and rounded once (no contraction: __dmul_rn / __dadd_rn);
// the overlap set of the initial pose.
#include "rf_common.cuh"

#define RF_PSO_OMEGA 0.7298
#define RF_PSO_C 1.49618

__device__ __forceinline__ void rf_clamp_store(double d[6], float* out) {
  const double n = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2])));
  if (n > 0.95) {
    const double sc = __ddiv_rn(0.95, n);
#pragma unroll
    for (int a = 0; a < 3; ++a) d[a] = __dmul_rn(d[a], sc);
  }
#pragma unroll
  for (int a = 0; a < 6; ++a) out[a] = (float)d[a];
}

struct Sigma6 { float s[6]; };

// Eq. (12): delta_out_i = clamp(delta_in_{a(i)} + sigma (.) z_i)
__global__ void k_propose(const float* __restrict__ din, const int* __restrict__ anc, Sigma6 sg, const float* __restrict__ z, int N,
                          float* __restrict__ dout) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int a0 = anc ? anc[i] : i;
  double d[6];
#pragma unroll
  for (int a = 0; a < 6; ++a) d[a] = __dadd_rn((double)din[6 * (size_t)a0 + a], __dmul_rn((double)sg.s[a], (double)z[6 * (size_t)i + a]));
  rf_clamp_store(d, dout + 6 * (size_t)i);
}

// Systematic resampling (B1) in ONE CTA of 1024 threads: normalised weights w_i / sum(w) accumulated in fp64 (per-thread
// runs of consecutive particles, then a scan of the run totals), then every slot u_m = (m + u) / N finds the first particle
// whose cumulative weight exceeds it by binary search.
#define RS_THREADS 1024
__global__ void __launch_bounds__(RS_THREADS) k_resample(const float* __restrict__ w, int N, double u, double* __restrict__ C,
                                                         int* __restrict__ anc) {
  __shared__ double part[RS_THREADS];
  __shared__ double total;
  const int t = threadIdx.x;
  const int per = (N + RS_THREADS - 1) / RS_THREADS;
  const int lo = min(N, t * per), hi = min(N, lo + per);
  double s = 0.0;
  for (int i = lo; i < hi; ++i) s += (double)w[i];
  part[t] = s;
  __syncthreads();
  if (t == 0) { double tot = 0.0; for (int q = 0; q < RS_THREADS; ++q) tot += part[q]; total = tot; }
  __syncthreads();
  const double tot = total;
  // cumulative normalised weight: runs again, each term divided as the definition states
  s = 0.0;
  for (int i = lo; i < hi; ++i) s += (double)w[i] / tot;
  __syncthreads();
  part[t] = s;
  __syncthreads();
  if (t == 0) { double run = 0.0; for (int q = 0; q < RS_THREADS; ++q) { const double x = part[q]; part[q] = run; run += x; } }
  __syncthreads();
  double run = part[t];
  for (int i = lo; i < hi; ++i) { run += (double)w[i] / tot; C[i] = run; }
  __syncthreads();
  if (t == 0) C[N - 1] = 2.0;                 // the last particle closes the unit interval whatever the rounding
  __threadfence_block();
  __syncthreads();
  for (int m = t; m < N; m += RS_THREADS) {
    const double um = ((double)m + u) / (double)N;
    int a = 0, b = N - 1;                     // first i with C_i > um
    while (a < b) { const int mid = (a + b) >> 1; if (C[mid] > um) b = mid; else a = mid + 1; }
    anc[m] = a;
  }
}

// PSO move (B2): v <- omega v + c1 a (p - x) + c2 b (g - x);  x <- clamp(x + v)
__global__ void k_pso_move(float* __restrict__ x, float* __restrict__ v, const float* __restrict__ pbest, const float* __restrict__ gbest,
                           const float* __restrict__ ua, const float* __restrict__ ub, int N) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  double d[6];
#pragma unroll
  for (int a = 0; a < 6; ++a) {
    const size_t q = 6 * (size_t)i + a;
    const double xi = (double)x[q];
    const double t1 = __dmul_rn(RF_PSO_OMEGA, (double)v[q]);
    const double t2 = __dmul_rn(__dmul_rn(RF_PSO_C, (double)ua[q]), __dadd_rn((double)pbest[q], -xi));
    const double t3 = __dmul_rn(__dmul_rn(RF_PSO_C, (double)ub[q]), __dadd_rn((double)gbest[a], -xi));
    const float vn = (float)__dadd_rn(__dadd_rn(t1, t2), t3);
    v[q] = vn;
    d[a] = __dadd_rn(xi, (double)vn);
  }
  rf_clamp_store(d, x + 6 * (size_t)i);
}

// Best-so-far bookkeeping in ONE CTA: personal bests (optional, strict improvement) and the swarm / run best
// (gbest[8] = 6 coordinates, fitness, index): the highest fitness of this step, lowest index among equals (A18),
// replaces the holder only if strictly better.
__global__ void __launch_bounds__(1024) k_best(const float* __restrict__ fit, const float* __restrict__ x, int N, float* __restrict__ pbest,
                                               float* __restrict__ pbest_fit, int first, float* __restrict__ gbest) {
  __shared__ float sv[32];
  __shared__ int si[32];
  float bv = -INFINITY; int bi = 0x7fffffff;
  for (int i = threadIdx.x; i < N; i += blockDim.x) {
    const float f = fit[i];
    if (pbest && (first || f > pbest_fit[i])) {
      pbest_fit[i] = f;
#pragma unroll
      for (int a = 0; a < 6; ++a) pbest[6 * (size_t)i + a] = x[6 * (size_t)i + a];
    }
    if (f > bv || (f == bv && i < bi) || bi == 0x7fffffff) { bv = f; bi = i; }      // ascending i per thread
  }
  for (int o = 16; o; o >>= 1) {
    const float ov = __shfl_xor_sync(0xffffffffu, bv, o); const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
    if (oi != 0x7fffffff && (bi == 0x7fffffff || ov > bv || (ov == bv && oi < bi))) { bv = ov; bi = oi; }
  }
  if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = bv; si[threadIdx.x >> 5] = bi; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int q = 1; q < (int)(blockDim.x >> 5); ++q)
      if (si[q] != 0x7fffffff && (bi == 0x7fffffff || sv[q] > bv || (sv[q] == bv && si[q] < bi))) { bv = sv[q]; bi = si[q]; }
    if (bi != 0x7fffffff && (first || bv > gbest[6])) {
      for (int a = 0; a < 6; ++a) gbest[a] = x[6 * (size_t)bi + a];
      gbest[6] = bv; gbest[7] = (float)bi;
    }
  }
}

extern "C" int rf_baseline_propose(rf_volume* v, const float* delta_in_dev, const int32_t* ancestors_dev_or_null, const float sigma[6],
                                   const float* normals_dev, int32_t N, float* delta_out_dev) {
  RF_ARG(v && delta_in_dev && sigma && normals_dev && delta_out_dev && N > 0, "rf_baseline_propose: bad argument");
  RF_ARG(delta_in_dev != delta_out_dev, "rf_baseline_propose: in place is not supported (ancestors are read while slots are written)");
  Sigma6 sg;
  for (int a = 0; a < 6; ++a) sg.s[a] = sigma[a];
  k_propose<<<(N + 255) / 256, 256, 0, v->stream>>>(delta_in_dev, ancestors_dev_or_null, sg, normals_dev, N, delta_out_dev);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  return RF_OK;
}

extern "C" int rf_baseline_resample(rf_volume* v, const float* fitness_dev, int32_t N, double u, int32_t* ancestors_out_dev) {
  RF_ARG(v && fitness_dev && ancestors_out_dev && N > 0 && u >= 0.0 && u < 1.0, "rf_baseline_resample: bad argument");
  int rc = rf_ensure((void**)&v->base_scratch, &v->base_cap, (size_t)N * sizeof(double));
  if (rc != RF_OK) return rc;
  k_resample<<<1, RS_THREADS, 0, v->stream>>>(fitness_dev, N, u, (double*)v->base_scratch, ancestors_out_dev);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  return RF_OK;
}

extern "C" int rf_baseline_pso_move(rf_volume* v, float* x_dev, float* v_dev, const float* pbest_dev, const float* gbest_dev,
                                    const float* ua_dev, const float* ub_dev, int32_t N) {
  RF_ARG(v && x_dev && v_dev && pbest_dev && gbest_dev && ua_dev && ub_dev && N > 0, "rf_baseline_pso_move: bad argument");
  k_pso_move<<<(N + 255) / 256, 256, 0, v->stream>>>(x_dev, v_dev, pbest_dev, gbest_dev, ua_dev, ub_dev, N);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  return RF_OK;
}

extern "C" int rf_baseline_best(rf_volume* v, const float* fitness_dev, const float* x_dev, int32_t N, float* pbest_dev_or_null,
                                float* pbest_fit_dev_or_null, int32_t first, float* gbest_dev) {
  RF_ARG(v && fitness_dev && x_dev && gbest_dev && N > 0, "rf_baseline_best: bad argument");
  RF_ARG((pbest_dev_or_null == nullptr) == (pbest_fit_dev_or_null == nullptr), "rf_baseline_best: pbest and pbest_fit go together");
  k_best<<<1, 1024, 0, v->stream>>>(fitness_dev, x_dev, N, pbest_dev_or_null, pbest_fit_dev_or_null, first, gbest_dev);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  return RF_OK;
}

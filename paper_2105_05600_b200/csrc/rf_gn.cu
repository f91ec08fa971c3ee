// rf_gn.cu -- Gauss-Newton minimisation of Eq. (4) on the fused volume (the SDF tracker of [Bylow 2013] the
// paper compares its optimiser with; reading GN1 in DESIGN.md).
//
// Same objective and sample rule as the fitness kernel: E(T) = sum over the valid points of psi(R x + t)^2, a point being
// valid when all 8 corners of its interpolation cell are observed.  One iteration is two launches and no host round trip:
//   k_gn_accumulate  one thread per point (grid-stride): residual psi, analytic gradient of the trilinear interpolant,
//                    J = [p x grad ; grad]; the 21 + 6 + 2 sums (upper triangle of J J^T, J psi, psi^2, count) are reduced
//                    lane -> warp -> CTA in a fixed order and written as one row of partials per CTA (no atomics);
//   k_gn_solve       one CTA: folds the partial rows in a fixed order, solves the 6x6 system (partial pivoting), applies the
//                    left-multiplied twist (R <- exp(omega) R, t <- exp(omega) t + v), records the trace row and raises the
//                    stop flag (|xi| < 1e-9, fewer than 6 points, or a singular system) that turns later launches into no-ops.
// Everything is fp64: the path is one pose over <= 3e5 points (a few hundred fp64 operations each), five orders of magnitude
// below the fitness kernel's work, and fp64 keeps the normal equations comparable with the oracle's to rounding order.
// The TSDF is read directly from the bricked volume (8 scalar loads per point), so no gather atlas is needed.
#include <algorithm>
#include <mutex>

#include "rf_common.cuh"

#define GN_THREADS 256
#define GN_VALS 29          // 21 upper-triangular entries of A (row-major), 6 of b, the cost, the number of points
#define GN_ROW 32           // doubles per partial row
#define GN_MAX_CTAS (148 * 4)

struct GnState {
  double T[12];
  int done, iters_run;
};

template <typename T> __device__ __forceinline__ double gn_voxel(const T* tsdf, unsigned off);
template <> __device__ __forceinline__ double gn_voxel<__half>(const __half* tsdf, unsigned off) { return (double)__half2float(tsdf[off]); }
template <> __device__ __forceinline__ double gn_voxel<float>(const float* tsdf, unsigned off) { return (double)tsdf[off]; }

template <typename T>
__global__ void __launch_bounds__(GN_THREADS) k_gn_accumulate(const T* __restrict__ tsdf, VolGeom g, const float4* __restrict__ pts,
                                                              int M, const GnState* __restrict__ st, double* __restrict__ partial,
                                                              const unsigned* __restrict__ slot_of) {
  if (st->done) return;
  double Tm[12];
#pragma unroll
  for (int a = 0; a < 12; ++a) Tm[a] = st->T[a];
  double acc[GN_VALS];
#pragma unroll
  for (int a = 0; a < GN_VALS; ++a) acc[a] = 0.0;
  const double vs = (double)g.vs;
  for (int i = blockIdx.x * GN_THREADS + threadIdx.x; i < M; i += gridDim.x * GN_THREADS) {
    const float4 x = __ldg(pts + i);
    if (x.w == 0.f) continue;
    double p[3], f[3];
    int i0[3];
    bool ok = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      p[a] = Tm[4 * a] * (double)x.x + Tm[4 * a + 1] * (double)x.y + Tm[4 * a + 2] * (double)x.z + Tm[4 * a + 3];
      const double gc = (p[a] - (double)g.origin[a]) / vs - 0.5;
      const double fl = floor(gc);
      f[a] = gc - fl;
      ok = ok && fl >= 0.0 && fl + 1.0 <= (double)(g.dims[a] - 1);       // also rejects NaN / huge coordinates
      i0[a] = ok ? (int)fl : 0;
    }
    if (!ok) continue;
    double v[8];
    bool seen = true;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      const int cx = i0[0] + (c & 1), cy = i0[1] + ((c >> 1) & 1), cz = i0[2] + (c >> 2);
      if (slot_of) {                                                     // sparse volume: a brick without a slot is unobserved
        const unsigned slot = slot_of[rf_brick_index(cx, cy, cz, g.bdims[0], g.bdims[1])];
        v[c] = slot == RF_NO_SLOT ? __longlong_as_double(0x7ff8000000000000ll) : gn_voxel<T>(tsdf, slot * RF_BRICK_VOX + rf_in_brick(cx, cy, cz));
      } else {
        v[c] = gn_voxel<T>(tsdf, rf_brick_offset(cx, cy, cz, g.bdims[0], g.bdims[1]));
      }
      seen = seen && v[c] == v[c];                                       // NaN = unobserved
    }
    if (!seen) continue;
    double psi = 0, gr[3] = {0, 0, 0};
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      const int cx = c & 1, cy = (c >> 1) & 1, cz = c >> 2;
      const double wx = cx ? f[0] : 1 - f[0], wy = cy ? f[1] : 1 - f[1], wz = cz ? f[2] : 1 - f[2];
      psi += wx * wy * wz * v[c];
      gr[0] += (cx ? 1.0 : -1.0) * wy * wz * v[c];
      gr[1] += wx * (cy ? 1.0 : -1.0) * wz * v[c];
      gr[2] += wx * wy * (cz ? 1.0 : -1.0) * v[c];
    }
    gr[0] /= vs; gr[1] /= vs; gr[2] /= vs;
    const double J[6] = {p[1] * gr[2] - p[2] * gr[1], p[2] * gr[0] - p[0] * gr[2], p[0] * gr[1] - p[1] * gr[0], gr[0], gr[1], gr[2]};
    int k = 0;
#pragma unroll
    for (int r = 0; r < 6; ++r)
#pragma unroll
      for (int c = r; c < 6; ++c) acc[k++] += J[r] * J[c];
#pragma unroll
    for (int r = 0; r < 6; ++r) acc[21 + r] += J[r] * psi;
    acc[27] += psi * psi;
    acc[28] += 1.0;
  }
  // lane -> warp -> CTA, every step in a fixed order
  __shared__ double red[GN_THREADS / 32][GN_ROW];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int a = 0; a < GN_VALS; ++a) {
    double s = acc[a];
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) red[warp][a] = s;
  }
  __syncthreads();
  if (threadIdx.x < GN_VALS) {
    double s = 0.0;
    for (int w = 0; w < GN_THREADS / 32; ++w) s += red[w][threadIdx.x];
    partial[(size_t)blockIdx.x * GN_ROW + threadIdx.x] = s;
  }
}

__device__ bool gn_solve6(double* A, double* b, double* x) {
  for (int c = 0; c < 6; ++c) {
    int piv = c;
    for (int r = c + 1; r < 6; ++r) if (fabs(A[6 * r + c]) > fabs(A[6 * piv + c])) piv = r;
    if (!(fabs(A[6 * piv + c]) > 1e-300)) return false;
    if (piv != c) {
      for (int k = 0; k < 6; ++k) { const double t = A[6 * c + k]; A[6 * c + k] = A[6 * piv + k]; A[6 * piv + k] = t; }
      const double t = b[c]; b[c] = b[piv]; b[piv] = t;
    }
    for (int r = c + 1; r < 6; ++r) {
      const double m = A[6 * r + c] / A[6 * c + c];
      for (int k = c; k < 6; ++k) A[6 * r + k] -= m * A[6 * c + k];
      b[r] -= m * b[c];
    }
  }
  for (int r = 5; r >= 0; --r) {
    double s = b[r];
    for (int k = r + 1; k < 6; ++k) s -= A[6 * r + k] * x[k];
    x[r] = s / A[6 * r + r];
  }
  return true;
}

// exp of a rotation vector: R = I + (sin th / th) [w]x + ((1 - cos th) / th^2) [w]x^2 (series below 1e-8 rad)
__device__ void gn_rodrigues(const double* w, double* R) {
  const double th = sqrt(w[0] * w[0] + w[1] * w[1] + w[2] * w[2]);
  double a, b;
  if (th < 1e-8) { a = 1.0 - th * th / 6.0; b = 0.5 - th * th / 24.0; }
  else { a = sin(th) / th; b = (1.0 - cos(th)) / (th * th); }
  const double K[9] = {0, -w[2], w[1], w[2], 0, -w[0], -w[1], w[0], 0};
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      double k2 = 0;
      for (int k = 0; k < 3; ++k) k2 += K[3 * i + k] * K[3 * k + j];
      R[3 * i + j] = (i == j ? 1.0 : 0.0) + a * K[3 * i + j] + b * k2;
    }
}

__global__ void __launch_bounds__(GN_ROW * 32) k_gn_solve(GnState* __restrict__ st, const double* __restrict__ partial, int nctas,
                                                           rf_gn_row* __restrict__ rows) {
  if (st->done) return;
  __shared__ double tot[GN_ROW];
  const int val = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double s = 0.0;
  if (val < GN_VALS)
    for (int c = lane; c < nctas; c += 32) s += partial[(size_t)c * GN_ROW + val];
  for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) tot[val] = s;
  __syncthreads();
  if (threadIdx.x != 0) return;
  double A[36], b[6], rhs[6], xi[6];
  int k = 0;
  for (int r = 0; r < 6; ++r)
    for (int c = r; c < 6; ++c) { A[6 * r + c] = tot[k]; A[6 * c + r] = tot[k]; ++k; }
  for (int r = 0; r < 6; ++r) { b[r] = tot[21 + r]; rhs[r] = -b[r]; }
  const int it = st->iters_run;
  rf_gn_row& row = rows[it];
  row.cost = tot[27]; row.n = (int)tot[28]; row.pad = 0; row.step_norm = 0.0;
  for (int a = 0; a < 36; ++a) row.A[a] = A[a];
  for (int a = 0; a < 6; ++a) row.b[a] = b[a];
  st->iters_run = it + 1;
  if (row.n < 6 || !gn_solve6(A, rhs, xi)) { st->done = 1; return; }
  double Rw[9], Tn[12];
  gn_rodrigues(xi, Rw);
  const double* T = st->T;
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) Tn[4 * i + j] = Rw[3 * i] * T[j] + Rw[3 * i + 1] * T[4 + j] + Rw[3 * i + 2] * T[8 + j];
    Tn[4 * i + 3] = Rw[3 * i] * T[3] + Rw[3 * i + 1] * T[7] + Rw[3 * i + 2] * T[11] + xi[3 + i];
  }
  for (int a = 0; a < 12; ++a) st->T[a] = Tn[a];
  double nn = 0;
  for (int r = 0; r < 6; ++r) nn += xi[r] * xi[r];
  row.step_norm = sqrt(nn);
  if (row.step_norm < 1e-9) st->done = 1;
}

extern "C" int rf_gn_track(rf_volume* v, const float* points_dev, int32_t M, const double pose_in[12], int32_t iters,
                           double pose_out[12], rf_gn_row* rows_out_or_null, int32_t* iters_run_out) {
  RF_ARG(v && (points_dev || M == 0) && pose_in && pose_out && iters_run_out, "rf_gn_track: NULL argument");
  RF_ARG(M >= 0 && iters >= 0 && iters <= 1024, "rf_gn_track: M must be >= 0 and iters in [0, 1024]");
  RF_ARG(((uintptr_t)points_dev & 15) == 0, "rf_gn_track: points_dev must be 16-byte aligned");
  const int nctas = std::max(1, std::min(GN_MAX_CTAS, (M + GN_THREADS - 1) / GN_THREADS));
  const size_t state_b = 256, rows_b = ((size_t)std::max(iters, 1) * sizeof(rf_gn_row) + 255) / 256 * 256;
  const size_t need = state_b + rows_b + (size_t)nctas * GN_ROW * sizeof(double);
  if (rf_ensure(&v->base_scratch, &v->base_cap, need) != RF_OK) return RF_ERR_CUDA;
  char* base = (char*)v->base_scratch;
  GnState* st = (GnState*)base;
  rf_gn_row* rows = (rf_gn_row*)(base + state_b);
  double* partial = (double*)(base + state_b + rows_b);
  GnState h;
  memcpy(h.T, pose_in, sizeof(h.T));
  h.done = 0; h.iters_run = 0;
  RF_CUDA(cudaMemcpyAsync(st, &h, sizeof(h), cudaMemcpyHostToDevice, v->stream));
  RF_CUDA(cudaStreamSynchronize(v->stream));                       // h lives on this stack frame
  for (int k = 0; k < iters; ++k) {
    if (v->g.dtype == RF_F16_W8)
      k_gn_accumulate<__half><<<nctas, GN_THREADS, 0, v->stream>>>((const __half*)v->tsdf, v->g, (const float4*)points_dev, M, st, partial, v->slot_of);
    else
      k_gn_accumulate<float><<<nctas, GN_THREADS, 0, v->stream>>>((const float*)v->tsdf, v->g, (const float4*)points_dev, M, st, partial, v->slot_of);
    k_gn_solve<<<1, GN_ROW * 32, 0, v->stream>>>(st, partial, nctas, rows);
    RF_LAUNCHED(2);
  }
  RF_CUDA(cudaGetLastError());
  RF_CUDA(cudaMemcpyAsync(&h, st, sizeof(h), cudaMemcpyDeviceToHost, v->stream));
  RF_CUDA(cudaStreamSynchronize(v->stream));
  memcpy(pose_out, h.T, sizeof(h.T));
  *iters_run_out = h.iters_run;
  if (rows_out_or_null && h.iters_run > 0)
    RF_CUDA(cudaMemcpy(rows_out_or_null, rows, (size_t)h.iters_run * sizeof(rf_gn_row), cudaMemcpyDeviceToHost));
  return RF_OK;
}

// ------------------------------------------------------------------------------------------------------------------------
// rf_gn_track_noalloc: the same iteration (the same two kernels, the same launch shapes, hence bit-identical results) for
// callers that may not allocate: code under stream capture, tight serving loops, harnesses that forbid cudaMalloc.
// The scratch of the run (state, one trace row per iteration, one row of partial sums per CTA) lives in ONE file-scope
// device array of fixed size, which every GPU that loads the library holds until the process exits:
//   256 B state + 64 trace rows of 360 B (23040 B) + 592 partial rows of 32 doubles (151552 B) = 174848 B.
// The limit that follows is RF_GN_NOALLOC_MAX_ITERS = 64 iterations per call; the number of points is not limited (the
// grid is capped at 592 CTAs for any M).  Every call on a device shares the array and finds the last call's contents in
// it: the state (pose, stop flag, iteration counter) is re-initialised by k_gn_init at the start of each call, every
// partial row a solve reads was written by the accumulate launch just before it, and only the trace rows of this call are
// read back, so nothing stale is ever consumed -- but two calls that overlap on the GPU (different streams, different
// volumes, different host threads) race on the array and must be serialised by the caller.
// In host code `g_gn_scratch` is only a stand-in for the symbol: the device address is taken once per device with
// cudaGetSymbolAddress (with that device current) and that pointer is what the kernels get.
#define GN_NOALLOC_STATE_B 256
#define GN_NOALLOC_ROWS_B ((RF_GN_NOALLOC_MAX_ITERS * sizeof(rf_gn_row) + 255) / 256 * 256)
#define GN_NOALLOC_BYTES (GN_NOALLOC_STATE_B + GN_NOALLOC_ROWS_B + (size_t)GN_MAX_CTAS * GN_ROW * sizeof(double))
static __device__ __align__(256) unsigned char g_gn_scratch[GN_NOALLOC_BYTES];

#define GN_MAX_DEVICES 64
static std::mutex g_gn_scratch_mu;
static void* g_gn_scratch_ptr[GN_MAX_DEVICES];          // device address of g_gn_scratch on device i (NULL: not asked yet)

struct GnPose { double T[12]; };
__global__ void k_gn_init(GnState* __restrict__ st, GnPose p) {
  if (threadIdx.x < 12) st->T[threadIdx.x] = p.T[threadIdx.x];
  if (threadIdx.x == 0) { st->done = 0; st->iters_run = 0; }
}

// the scratch array's address on the current device (set-up: once per device)
static int gn_scratch_here(int dev, void** out) {
  std::lock_guard<std::mutex> lock(g_gn_scratch_mu);
  if (!g_gn_scratch_ptr[dev]) {
    void* p = nullptr;
    RF_CUDA(cudaGetSymbolAddress(&p, g_gn_scratch));
    RF_ARG(p != nullptr, "rf_gn_track_noalloc: cudaGetSymbolAddress returned NULL");
    g_gn_scratch_ptr[dev] = p;
  }
  *out = g_gn_scratch_ptr[dev];
  return RF_OK;
}

extern "C" int64_t rf_gn_noalloc_scratch_bytes(void) { return (int64_t)GN_NOALLOC_BYTES; }

extern "C" int rf_gn_track_noalloc(rf_volume* v, const float* points_dev, int32_t M, const double pose_in[12], int32_t iters,
                                   double pose_out[12], rf_gn_row* rows_out_or_null, int32_t* iters_run_out) {
  RF_ARG(v && (points_dev || M == 0) && pose_in && pose_out && iters_run_out, "rf_gn_track_noalloc: NULL argument");
  RF_ARG(M >= 0 && iters >= 0, "rf_gn_track_noalloc: M and iters must be >= 0");
  RF_ARG(iters <= RF_GN_NOALLOC_MAX_ITERS,
         "rf_gn_track_noalloc: iters exceeds RF_GN_NOALLOC_MAX_ITERS (64), the size of the static trace; use rf_gn_track");
  RF_ARG(((uintptr_t)points_dev & 15) == 0, "rf_gn_track_noalloc: points_dev must be 16-byte aligned");
  int dev = -1;
  RF_CUDA(cudaGetDevice(&dev));
  RF_ARG(dev >= 0 && dev < GN_MAX_DEVICES, "rf_gn_track_noalloc: device ordinal beyond 63");
  {
    // the static array is per device: the device that is current must be the one that holds the volume
    cudaPointerAttributes attr;
    RF_CUDA(cudaPointerGetAttributes(&attr, v->tsdf));
    RF_ARG(attr.device == dev, "rf_gn_track_noalloc: the volume's device is not the current device");
  }
  void* scratch = nullptr;
  int rc = gn_scratch_here(dev, &scratch);
  if (rc != RF_OK) return rc;
  char* base = (char*)scratch;
  GnState* st = (GnState*)base;
  rf_gn_row* rows = (rf_gn_row*)(base + GN_NOALLOC_STATE_B);
  double* partial = (double*)(base + GN_NOALLOC_STATE_B + GN_NOALLOC_ROWS_B);
  const int nctas = std::max(1, std::min(GN_MAX_CTAS, (M + GN_THREADS - 1) / GN_THREADS));     // as rf_gn_track
  GnPose p0;
  memcpy(p0.T, pose_in, sizeof(p0.T));
  k_gn_init<<<1, 32, 0, v->stream>>>(st, p0);             // clears what must start at zero (stop flag, iteration counter)
  RF_LAUNCHED(1);
  for (int k = 0; k < iters; ++k) {
    if (v->g.dtype == RF_F16_W8)
      k_gn_accumulate<__half><<<nctas, GN_THREADS, 0, v->stream>>>((const __half*)v->tsdf, v->g, (const float4*)points_dev, M, st, partial, v->slot_of);
    else
      k_gn_accumulate<float><<<nctas, GN_THREADS, 0, v->stream>>>((const float*)v->tsdf, v->g, (const float4*)points_dev, M, st, partial, v->slot_of);
    k_gn_solve<<<1, GN_ROW * 32, 0, v->stream>>>(st, partial, nctas, rows);
    RF_LAUNCHED(2);
  }
  RF_CUDA(cudaGetLastError());
  GnState h;
  RF_CUDA(cudaMemcpyAsync(&h, st, sizeof(h), cudaMemcpyDeviceToHost, v->stream));
  RF_CUDA(cudaStreamSynchronize(v->stream));
  memcpy(pose_out, h.T, sizeof(h.T));
  *iters_run_out = h.iters_run;
  if (rows_out_or_null && h.iters_run > 0) {
    RF_CUDA(cudaMemcpyAsync(rows_out_or_null, rows, (size_t)h.iters_run * sizeof(rf_gn_row), cudaMemcpyDeviceToHost, v->stream));
    RF_CUDA(cudaStreamSynchronize(v->stream));
  }
  return RF_OK;
}

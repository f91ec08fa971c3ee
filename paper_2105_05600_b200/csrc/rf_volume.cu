// rf_volume.cu -- volume life cycle, upload / download (step a7), error plumbing.
#include "rf_common.cuh"
#include <string.h>
#include <stdlib.h>
#include <limits>

static thread_local std::string g_err;
void rf_set_error(const std::string& s) { g_err = s; }
int rf_cuda_fail(cudaError_t e, const char* what) {
  g_err = std::string(what) + ": " + cudaGetErrorString(e);
  return e == cudaErrorMemoryAllocation ? RF_ERR_OOM : RF_ERR_CUDA;
}
extern "C" const char* rf_last_error(void) { return g_err.c_str(); }
extern "C" int rf_version(void) { return 100; }

long long g_rf_launches = 0;
thread_local int t_rf_capturing = 0;
thread_local long long t_rf_captured = 0;
extern "C" int64_t rf_launch_count(void) { return (int64_t)__atomic_load_n(&g_rf_launches, __ATOMIC_RELAXED); }

// ---- optional per-kernel timing: event pairs on the volume's stream, folded into sums after a sync ----
static void prof_event(rf_volume* v, int which) {
  if (v->prof_used[which] >= v->prof_cap[which]) {
    const int ncap = v->prof_cap[which] ? v->prof_cap[which] * 2 : 256;
    cudaEvent_t* ne = new cudaEvent_t[ncap];
    for (int i = 0; i < ncap; ++i) { if (i < v->prof_cap[which]) ne[i] = v->prof_ev[which][i]; else cudaEventCreate(&ne[i]); }
    delete[] v->prof_ev[which];
    v->prof_ev[which] = ne; v->prof_cap[which] = ncap;
  }
  cudaEventRecord(v->prof_ev[which][v->prof_used[which]++], v->stream);
}
void rf_prof_begin(rf_volume* v, int which) { if (v->prof_on) prof_event(v, which); }
void rf_prof_end(rf_volume* v, int which) { if (v->prof_on) prof_event(v, which); }
void rf_prof_collect(rf_volume* v) {       // call only after the stream has been synchronised
  for (int w = 0; w < RF_PROF_SLOTS; ++w) {
    for (int i = 0; i + 1 < v->prof_used[w]; i += 2) {
      float ms = 0;
      if (cudaEventElapsedTime(&ms, v->prof_ev[w][i], v->prof_ev[w][i + 1]) == cudaSuccess) {
        v->prof_ms[w] += ms; v->prof_launches[w] += 1;
        if (v->prof_each_n[w] >= v->prof_each_cap[w]) {
          const int ncap = v->prof_each_cap[w] ? 2 * v->prof_each_cap[w] : 1024;
          float* ne = (float*)realloc(v->prof_each[w], (size_t)ncap * sizeof(float));
          if (ne) { v->prof_each[w] = ne; v->prof_each_cap[w] = ncap; }
        }
        if (v->prof_each_n[w] < v->prof_each_cap[w]) v->prof_each[w][v->prof_each_n[w]++] = ms;
      }
    }
    v->prof_used[w] = 0;
  }
}
extern "C" int rf_profile_enable(rf_volume* v, int32_t on) {
  RF_ARG(v, "rf_profile_enable: NULL volume");
  RF_CUDA(cudaStreamSynchronize(v->stream));
  rf_prof_collect(v);
  v->prof_on = on ? 1 : 0;
  return RF_OK;
}
extern "C" int rf_profile_read(rf_volume* v, int32_t which, double* ms_out, int64_t* launches_out) {
  RF_ARG(v && ms_out && launches_out && which >= 0 && which < RF_PROF_SLOTS, "rf_profile_read: bad argument");
  RF_CUDA(cudaStreamSynchronize(v->stream));
  rf_prof_collect(v);
  *ms_out = v->prof_ms[which]; *launches_out = v->prof_launches[which];
  v->prof_ms[which] = 0; v->prof_launches[which] = 0;
  v->prof_each_n[which] = 0;
  return RF_OK;
}
extern "C" int rf_profile_read_launches(rf_volume* v, int32_t which, float* ms_each_out, int32_t cap, int32_t* n_out) {
  RF_ARG(v && ms_each_out && n_out && cap >= 0 && which >= 0 && which < RF_PROF_SLOTS, "rf_profile_read_launches: bad argument");
  RF_CUDA(cudaStreamSynchronize(v->stream));
  rf_prof_collect(v);
  const int n = v->prof_each_n[which] < cap ? v->prof_each_n[which] : cap;
  for (int i = 0; i < n; ++i) ms_each_out[i] = v->prof_each[which][i];
  *n_out = v->prof_each_n[which];
  return RF_OK;
}

int rf_ensure_acc(rf_volume* v, size_t total, cudaStream_t st) {
  if (total > v->acc_cap) {
    cudaFree(v->acc[0]); cudaFree(v->acc[1]); v->acc[0] = v->acc[1] = nullptr; v->acc_cap = 0;
    const size_t cap = total + 1024;
    RF_CUDA(cudaMalloc(&v->acc[0], cap * sizeof(unsigned long long)));
    RF_CUDA(cudaMalloc(&v->acc[1], cap * sizeof(unsigned long long)));
    v->acc_cap = cap;
    v->graph_valid = 0;                      // a captured graph holds the old pointers
  }
  // start every API call from zero: robust against a previous call that failed half-way
  RF_CUDA(cudaMemsetAsync(v->acc[0], 0, v->acc_cap * sizeof(unsigned long long), st));
  RF_CUDA(cudaMemsetAsync(v->acc[1], 0, v->acc_cap * sizeof(unsigned long long), st));
  RF_CUDA(cudaMemsetAsync(v->d_MO, 0, 4 * sizeof(int), st));
  return RF_OK;
}

int rf_ensure(void** p, size_t* cap, size_t need) {
  if (*cap >= need && *p) return RF_OK;
  if (*p) cudaFree(*p);
  *p = nullptr; *cap = 0;
  RF_CUDA(cudaMalloc(p, need));
  *cap = need;
  return RF_OK;
}

// ---- fill: every voxel unobserved (TSDF = quiet NaN, W = 0) ----
template <typename T> __device__ __forceinline__ T rf_nan();
template <> __device__ __forceinline__ float rf_nan<float>() { return __int_as_float(0x7fc00000); }
template <> __device__ __forceinline__ __half rf_nan<__half>() { return __ushort_as_half((unsigned short)0x7e00); }

template <typename T>
__global__ void k_reset(T* tsdf, uint8_t* weight, size_t n) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    tsdf[i] = rf_nan<T>();
    weight[i] = 0;
  }
}

extern "C" int rf_volume_reset(rf_volume* v) {
  RF_ARG(v, "rf_volume_reset: NULL volume");
  const int blocks = 148 * 8;
  if (v->g.dtype == RF_F16_W8) k_reset<__half><<<blocks, 256, 0, v->stream>>>((__half*)v->tsdf, v->weight, v->nvox);
  else k_reset<float><<<blocks, 256, 0, v->stream>>>((float*)v->tsdf, v->weight, v->nvox);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  if (v->pool_bricks) {
    // sparse: nothing is allocated any more; a brick is flagged for the atlas when it is allocated
    RF_CUDA(cudaMemsetAsync(v->slot_of, 0xff, v->nbricks * sizeof(unsigned), v->stream));
    RF_CUDA(cudaMemsetAsync(v->pool_used, 0, 4 * sizeof(unsigned), v->stream));
    RF_CUDA(cudaMemsetAsync(v->brick_dirty, 0, v->nbricks, v->stream));
  } else {
    // every brick of the gather atlas is now out of date
    RF_CUDA(cudaMemsetAsync(v->brick_dirty, 1, v->nbricks, v->stream));
  }
  v->atlas_stale = 1;
  return RF_OK;
}

extern "C" int rf_volume_create_ex(const int32_t dims[3], float voxel_size, float trunc, const rf_volume_opts* o,
                                   rf_volume** out) {
  RF_ARG(dims && out, "rf_volume_create: NULL argument");
  RF_ARG(dims[0] > 0 && dims[1] > 0 && dims[2] > 0, "rf_volume_create: dims must be positive");
  RF_ARG(dims[0] <= 8192 && dims[1] <= 8192 && dims[2] <= 8192, "rf_volume_create: at most 8192 voxels per axis");
  RF_ARG(voxel_size > 0.f && isfinite(voxel_size), "rf_volume_create: voxel_size must be positive");
  RF_ARG(trunc >= voxel_size && isfinite(trunc), "rf_volume_create: trunc must be >= voxel_size");
  rf_volume_opts opts; memset(&opts, 0, sizeof(opts)); opts.w_max = 255;
  if (o) opts = *o;
  if (opts.w_max == 0) opts.w_max = 255;
  RF_ARG(opts.dtype == RF_F32_W8 || opts.dtype == RF_F16_W8, "rf_volume_create: bad dtype");
  RF_ARG(opts.w_max >= 1 && opts.w_max <= 255, "rf_volume_create: w_max must be in 1..255");
  RF_ARG(opts.pool_bricks >= 0 && opts.pool_bricks <= (1 << 23) - 1, "rf_volume_create: pool_bricks must be in 0 .. 2^23 - 1");
  int dev = 0; cudaDeviceProp prop;
  RF_CUDA(cudaGetDevice(&dev));
  RF_CUDA(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10) { rf_set_error("rf_volume_create: device is not sm_100"); return RF_ERR_UNSUPPORTED; }
  rf_volume* v = new rf_volume();
  memset(v, 0, sizeof(*v));
  for (int a = 0; a < 3; ++a) {
    v->g.dims[a] = dims[a];
    v->g.bdims[a] = (dims[a] + RF_BRICK - 1) / RF_BRICK;
    v->g.origin[a] = opts.origin[a];
  }
  v->g.vs = voxel_size; v->g.trunc = trunc; v->g.inv_vs = (float)(1.0 / (double)voxel_size);
  v->g.dtype = opts.dtype; v->g.w_max = opts.w_max;
  v->stream = (cudaStream_t)opts.stream;
  v->nbricks = (size_t)v->g.bdims[0] * v->g.bdims[1] * v->g.bdims[2];
  v->pool_bricks = (unsigned)opts.pool_bricks;
  if (v->pool_bricks) {
    if (v->nbricks > (1ull << 25)) { delete v; rf_set_error("rf_volume_create: a sparse volume has at most 2^25 logical bricks"); return RF_ERR_INVALID_ARG; }
    v->nvox = (size_t)v->pool_bricks * RF_BRICK_VOX;
  } else {
    v->nvox = v->nbricks * RF_BRICK_VOX;
  }
  if (v->nvox > 0xfffffff0ull) { delete v; rf_set_error("rf_volume_create: more than 2^32 voxels"); return RF_ERR_INVALID_ARG; }
  const size_t esz = opts.dtype == RF_F16_W8 ? 2 : 4;
  cudaError_t e;
  if ((e = cudaMalloc(&v->tsdf, v->nvox * esz)) != cudaSuccess ||
      (e = cudaMalloc(&v->weight, v->nvox)) != cudaSuccess ||
      (e = cudaMalloc(&v->brick_list, v->nbricks * sizeof(unsigned))) != cudaSuccess ||
      (e = cudaMalloc(&v->brick_base, v->nbricks * sizeof(float4))) != cudaSuccess ||
      (e = cudaMalloc(&v->brick_count, 4 * sizeof(unsigned))) != cudaSuccess ||
      (v->pool_bricks && ((e = cudaMalloc(&v->slot_of, v->nbricks * sizeof(unsigned))) != cudaSuccess ||
                          (e = cudaMalloc(&v->brick_pslot, v->nbricks * sizeof(unsigned))) != cudaSuccess ||
                          (e = cudaMalloc(&v->brick_of, (size_t)v->pool_bricks * sizeof(unsigned))) != cudaSuccess ||
                          (e = cudaMalloc(&v->pool_used, 4 * sizeof(unsigned))) != cudaSuccess)) ||
      (e = cudaMalloc(&v->upd_count, sizeof(unsigned long long))) != cudaSuccess ||
      (e = cudaMalloc(&v->d_MO, 4 * sizeof(int))) != cudaSuccess ||
      (e = cudaMalloc(&v->brick_dirty, v->nbricks)) != cudaSuccess ||
      (e = cudaMalloc(&v->refresh_list, v->nbricks * sizeof(unsigned))) != cudaSuccess ||
      (e = cudaMalloc(&v->refresh_count, 4 * sizeof(unsigned))) != cudaSuccess ||
      (e = cudaMalloc(&v->init_dev, 512)) != cudaSuccess ||
      (e = cudaMallocHost(&v->init_host, 512)) != cudaSuccess ||
      (e = cudaStreamCreateWithFlags(&v->cap_stream, cudaStreamNonBlocking)) != cudaSuccess ||
      (e = cudaMalloc(&v->track, sizeof(TrackDev))) != cudaSuccess ||
      (e = cudaMalloc(&v->trace_dev, RF_MAX_ITERS * sizeof(rf_track_trace))) != cudaSuccess ||
      (e = cudaMallocHost(&v->track_host, sizeof(TrackDev))) != cudaSuccess ||
      (e = cudaMallocHost(&v->trace_host, RF_MAX_ITERS * sizeof(rf_track_trace))) != cudaSuccess) {
    rf_volume_destroy(v);
    return rf_cuda_fail(e, "rf_volume_create: allocation");
  }
  cudaMemsetAsync(v->upd_count, 0, sizeof(unsigned long long), v->stream);
  cudaMemsetAsync(v->refresh_count, 0, 4 * sizeof(unsigned), v->stream);
  int rc = rf_volume_reset(v);
  if (rc != RF_OK) { rf_volume_destroy(v); return rc; }
  *out = v;
  return RF_OK;
}

extern "C" int rf_volume_create(const int32_t dims[3], float voxel_size, float trunc, rf_volume** out) {
  return rf_volume_create_ex(dims, voxel_size, trunc, nullptr, out);
}

extern "C" int rf_volume_destroy(rf_volume* v) {
  if (!v) return RF_OK;
  cudaStreamSynchronize(v->stream);
  if (v->copy_stream) {
    cudaStreamSynchronize(v->copy_stream);
    cudaEventDestroy(v->pre_gate); cudaEventDestroy(v->pre_done[0]); cudaEventDestroy(v->pre_done[1]);
    cudaStreamDestroy(v->copy_stream);
  }
  cudaFree(v->pre_buf[0]); cudaFree(v->pre_buf[1]);
  cudaFree(v->tsdf); cudaFree(v->weight); cudaFree(v->depth_stage); cudaFree(v->depth_clean); cudaFree(v->tile_max);
  cudaFree(v->slot_of); cudaFree(v->brick_of); cudaFree(v->brick_pslot); cudaFree(v->pool_used);
  cudaFree(v->brick_list); cudaFree(v->brick_base); cudaFree(v->brick_count); cudaFree(v->upd_count);
  cudaFree(v->acc[0]); cudaFree(v->acc[1]); cudaFree(v->d_MO);
  cudaFree(v->atlas); cudaFree(v->brick_dirty); cudaFree(v->refresh_list); cudaFree(v->refresh_count);
  if (v->track_done) cudaEventDestroy(v->track_done);
  if (v->graph_exec) cudaGraphExecDestroy(v->graph_exec);
  if (v->cap_stream) cudaStreamDestroy(v->cap_stream);
  cudaFree(v->track); cudaFree(v->trace_dev); cudaFree(v->base_scratch); free(v->shard);
  for (int l = 0; l < 3; ++l) cudaFree(v->pts_raw[l]);
  cudaFree(v->init_dev);
  if (v->init_host) cudaFreeHost(v->init_host);
  if (v->track_host) cudaFreeHost(v->track_host);
  if (v->trace_host) cudaFreeHost(v->trace_host);
  for (int w = 0; w < RF_PROF_SLOTS; ++w) { for (int i = 0; i < v->prof_cap[w]; ++i) cudaEventDestroy(v->prof_ev[w][i]); delete[] v->prof_ev[w]; free(v->prof_each[w]); }
  delete v;
  return RF_OK;
}

// ---- dense <-> brick conversion, one z-slab of 8 at a time ----
template <typename T> __device__ __forceinline__ float rf_to_float(T v);
template <> __device__ __forceinline__ float rf_to_float<float>(float v) { return v; }
template <> __device__ __forceinline__ float rf_to_float<__half>(__half v) { return __half2float(v); }
template <typename T> __device__ __forceinline__ T rf_from_float(float v);
template <> __device__ __forceinline__ float rf_from_float<float>(float v) { return v; }
template <> __device__ __forceinline__ __half rf_from_float<__half>(float v) { return __float2half_rn(v); }

// dense slab: [nz][Y][X] floats starting at z0.  to_brick != 0: dense -> brick, else brick -> dense.
template <typename T>
__global__ void k_convert(T* tsdf, uint8_t* weight, float* dense_t, float* dense_w, VolGeom g, int z0, int nz,
                          int to_brick, const unsigned* __restrict__ slot_of) {
  const size_t n = (size_t)g.dims[0] * g.dims[1] * nz;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const int x = (int)(i % g.dims[0]);
    const int y = (int)((i / g.dims[0]) % g.dims[1]);
    const int z = z0 + (int)(i / ((size_t)g.dims[0] * g.dims[1]));
    unsigned off;
    if (slot_of) {                              // sparse: a brick without a slot is unobserved (upload: k_alloc_observed gave every
      const unsigned slot = slot_of[rf_brick_index(x, y, z, g.bdims[0], g.bdims[1])];     // brick with an observed voxel a slot)
      if (slot == RF_NO_SLOT) { if (!to_brick) { dense_t[i] = 1.0f; if (dense_w) dense_w[i] = 0.f; } continue; }
      off = slot * RF_BRICK_VOX + rf_in_brick(x, y, z);
    } else {
      off = rf_brick_offset(x, y, z, g.bdims[0], g.bdims[1]);
    }
    if (to_brick) {
      const float w = dense_w[i];
      const int wi = (int)fminf(fmaxf(w, 0.f), 255.f);
      weight[off] = (uint8_t)wi;
      tsdf[off] = wi > 0 ? rf_from_float<T>(dense_t[i]) : rf_nan<T>();
    } else {
      const int wi = weight[off];
      dense_t[i] = wi > 0 ? rf_to_float<T>(tsdf[off]) : 1.0f;
      if (dense_w) dense_w[i] = (float)wi;
    }
  }
}

// dense read-out of the box [lo, lo + size) (x fastest), dense or sparse volume
template <typename T>
__global__ void k_read_box(const T* __restrict__ tsdf, const uint8_t* __restrict__ weight, const unsigned* __restrict__ slot_of,
                           VolGeom g, int lx, int ly, int lz, int sx, int sy, int sz, float* __restrict__ out_t,
                           float* __restrict__ out_w) {
  const size_t n = (size_t)sx * sy * sz;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const int x = lx + (int)(i % sx), y = ly + (int)((i / sx) % sy), z = lz + (int)(i / ((size_t)sx * sy));
    unsigned b = rf_brick_index(x, y, z, g.bdims[0], g.bdims[1]);
    if (slot_of) b = slot_of[b];
    int wi = 0;
    float f = 1.0f;
    if (b != RF_NO_SLOT) {
      const size_t off = (size_t)b * RF_BRICK_VOX + rf_in_brick(x, y, z);
      wi = weight[off];
      if (wi > 0) f = rf_to_float<T>(tsdf[off]);
    }
    out_t[i] = f;
    if (out_w) out_w[i] = (float)wi;
  }
}

extern "C" int rf_volume_download_box(const rf_volume* v, const int32_t lo[3], const int32_t size[3], float* tsdf_out_dev,
                                      float* weight_out_dev_or_null) {
  RF_ARG(v && lo && size && tsdf_out_dev, "rf_volume_download_box: NULL argument");
  for (int a = 0; a < 3; ++a)
    RF_ARG(lo[a] >= 0 && size[a] > 0 && lo[a] + size[a] <= v->g.dims[a], "rf_volume_download_box: the box must lie inside the grid");
  const size_t n = (size_t)size[0] * size[1] * size[2];
  const int blocks = (int)min((size_t)148 * 8, (n + 255) / 256);
  if (v->g.dtype == RF_F16_W8)
    k_read_box<__half><<<blocks, 256, 0, v->stream>>>((const __half*)v->tsdf, v->weight, v->slot_of, v->g, lo[0], lo[1], lo[2], size[0], size[1], size[2], tsdf_out_dev, weight_out_dev_or_null);
  else
    k_read_box<float><<<blocks, 256, 0, v->stream>>>((const float*)v->tsdf, v->weight, v->slot_of, v->g, lo[0], lo[1], lo[2], size[0], size[1], size[2], tsdf_out_dev, weight_out_dev_or_null);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  return RF_OK;
}

// Upload into a sparse volume, one z-slab of bricks at a time: a brick of the slab with any observed voxel (W > 0) gets a slot.
// One thread per brick (a test / restore hook, not a hot path).
__global__ void k_alloc_observed(const float* __restrict__ dense_w, VolGeom g, int z0, int nz, unsigned* __restrict__ slot_of,
                                 unsigned* __restrict__ brick_of, unsigned* __restrict__ pool_used, unsigned pool_cap,
                                 uint8_t* __restrict__ brick_dirty) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= g.bdims[0] * g.bdims[1]) return;
  const int bx = t % g.bdims[0], by = t / g.bdims[0];
  bool any = false;
  for (int z = 0; z < nz && !any; ++z)
    for (int y = by * 8; y < min(by * 8 + 8, g.dims[1]) && !any; ++y)
      for (int x = bx * 8; x < min(bx * 8 + 8, g.dims[0]); ++x)
        if (dense_w[((size_t)z * g.dims[1] + y) * g.dims[0] + x] >= 1.0f) { any = true; break; }
  if (!any) return;
  const unsigned b = ((unsigned)(z0 >> 3) * (unsigned)g.bdims[1] + (unsigned)by) * (unsigned)g.bdims[0] + (unsigned)bx;
  if (slot_of[b] != RF_NO_SLOT) return;
  const unsigned slot = atomicAdd(pool_used, 1u);
  if (slot < pool_cap) { slot_of[b] = slot; brick_of[slot] = b; brick_dirty[b] = 1; }
  else atomicAdd(pool_used + 1, 1u);              // dropped: reported by rf_volume_pool_stats / rf_volume_upload
}

static int convert(const rf_volume* v, float* t_ext, float* w_ext, int ext_on_device, int to_brick) {
  const VolGeom& g = v->g;
  const size_t slab = (size_t)g.dims[0] * g.dims[1] * RF_BRICK;
  float *dt = nullptr, *dw = nullptr;
  if (!ext_on_device) {
    RF_CUDA(cudaMalloc(&dt, slab * sizeof(float)));
    cudaError_t e = cudaMalloc(&dw, slab * sizeof(float));
    if (e != cudaSuccess) { cudaFree(dt); return rf_cuda_fail(e, "convert scratch"); }
  }
  int rc = RF_OK;
  for (int z0 = 0; z0 < g.dims[2] && rc == RF_OK; z0 += RF_BRICK) {
    const int nz = min(RF_BRICK, g.dims[2] - z0);
    const size_t n = (size_t)g.dims[0] * g.dims[1] * nz;
    const size_t base = (size_t)g.dims[0] * g.dims[1] * z0;
    float* pt = ext_on_device ? t_ext + base : dt;
    float* pw = ext_on_device ? (w_ext ? w_ext + base : nullptr) : dw;
    cudaError_t e = cudaSuccess;
    if (!ext_on_device && to_brick) {
      e = cudaMemcpyAsync(dt, t_ext + base, n * sizeof(float), cudaMemcpyHostToDevice, v->stream);
      if (e == cudaSuccess) e = cudaMemcpyAsync(dw, w_ext + base, n * sizeof(float), cudaMemcpyHostToDevice, v->stream);
    }
    if (e == cudaSuccess && to_brick && v->pool_bricks) {
      const int nb = v->g.bdims[0] * v->g.bdims[1];
      k_alloc_observed<<<(nb + 127) / 128, 128, 0, v->stream>>>(pw, g, z0, nz, v->slot_of, v->brick_of, v->pool_used, v->pool_bricks, v->brick_dirty);
      e = cudaGetLastError();
    }
    if (e == cudaSuccess) {
      const int blocks = (int)min((size_t)148 * 8, (n + 255) / 256);
      if (g.dtype == RF_F16_W8) k_convert<__half><<<blocks, 256, 0, v->stream>>>((__half*)v->tsdf, v->weight, pt, pw, g, z0, nz, to_brick, v->slot_of);
      else k_convert<float><<<blocks, 256, 0, v->stream>>>((float*)v->tsdf, v->weight, pt, pw, g, z0, nz, to_brick, v->slot_of);
      e = cudaGetLastError();
    }
    if (e == cudaSuccess && !ext_on_device && !to_brick) {
      e = cudaMemcpyAsync(t_ext + base, dt, n * sizeof(float), cudaMemcpyDeviceToHost, v->stream);
      if (e == cudaSuccess && w_ext) e = cudaMemcpyAsync(w_ext + base, dw, n * sizeof(float), cudaMemcpyDeviceToHost, v->stream);
    }
    if (e == cudaSuccess && !ext_on_device) e = cudaStreamSynchronize(v->stream);   // scratch is reused per slab
    if (e != cudaSuccess) rc = rf_cuda_fail(e, "volume convert");
  }
  if (rc == RF_OK) { cudaError_t e = cudaStreamSynchronize(v->stream); if (e != cudaSuccess) rc = rf_cuda_fail(e, "volume convert sync"); }
  cudaFree(dt); cudaFree(dw);
  return rc;
}

extern "C" int rf_volume_download_ex(const rf_volume* v, float* tsdf_out, float* weight_out, int32_t on_device) {
  RF_ARG(v && tsdf_out, "rf_volume_download: NULL argument");
  return convert(v, tsdf_out, weight_out, on_device, 0);
}
extern "C" int rf_volume_download(const rf_volume* v, float* tsdf_out, float* weight_out) {
  return rf_volume_download_ex(v, tsdf_out, weight_out, 0);
}
extern "C" int rf_volume_upload(rf_volume* v, const float* tsdf, const float* weight) {
  RF_ARG(v && tsdf && weight, "rf_volume_upload: NULL argument");
  int rc = rf_volume_reset(v);
  if (rc != RF_OK) return rc;
  rc = convert(v, const_cast<float*>(tsdf), const_cast<float*>(weight), 0, 1);
  if (rc == RF_OK && v->pool_bricks) {
    // sparse: every brick with an observed voxel needed a slot
    int64_t st[4];
    rc = rf_volume_pool_stats(v, st);
    if (rc == RF_OK && st[2] > 0) { rf_set_error("rf_volume_upload: the pool is too small for the uploaded volume (bricks dropped)"); return RF_ERR_OOM; }
  }
  return rc;
}

extern "C" int rf_volume_pool_stats(rf_volume* v, int64_t out[4]) {
  RF_ARG(v && out, "rf_volume_pool_stats: NULL argument");
  out[0] = out[1] = (int64_t)v->nbricks; out[2] = out[3] = 0;
  if (!v->pool_bricks) return RF_OK;
  unsigned h[4] = {0, 0, 0, 0};
  RF_CUDA(cudaMemcpyAsync(h, v->pool_used, sizeof(h), cudaMemcpyDeviceToHost, v->stream));
  RF_CUDA(cudaStreamSynchronize(v->stream));
  out[0] = (int64_t)(h[0] < v->pool_bricks ? h[0] : v->pool_bricks);
  out[1] = (int64_t)v->pool_bricks;
  out[2] = (int64_t)h[1];
  return RF_OK;
}

// rf_surface.cu -- the surface point set of the fused TSDF ("marching cubes ... to point sets (no graphics API)",
// the reconstruction whose completeness / accuracy the paper measures; reading R-R2 in DESIGN.md).
//
// The vertex set of marching cubes: every grid edge between voxel a and its +x / +y / +z neighbour b whose two samples are
// both observed and lie on different sides of the surface (exactly one of psi_a, psi_b is > 0) carries one point, the zero of
// the straight line through the two samples.  One thread = one x-row of 8 voxels of a brick (one 128-bit TSDF load; the +y
// and +z rows are two more, the +x neighbour of the last voxel one scalar load); an unobserved sample holds NaN, which is
// on neither side.  Points are appended with one atomic per warp; the output order is not defined, each point carries its
// edge key 3 * (i + X (j + Y k)) + axis so that a caller can sort.
#include "rf_common.cuh"

template <typename T> struct SRow;
template <> struct SRow<__half> {
  static __device__ __forceinline__ void load(const __half* p, float* out) {
    const uint4 r = __ldg(reinterpret_cast<const uint4*>(p));
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const unsigned w = (&r.x)[e];
      out[2 * e] = __half2float(__ushort_as_half((unsigned short)(w & 0xffffu)));
      out[2 * e + 1] = __half2float(__ushort_as_half((unsigned short)(w >> 16)));
    }
  }
  static __device__ __forceinline__ float one(const __half* p) { return __half2float(*p); }
};
template <> struct SRow<float> {
  static __device__ __forceinline__ void load(const float* p, float* out) {
    const float4 a = __ldg(reinterpret_cast<const float4*>(p)), b = __ldg(reinterpret_cast<const float4*>(p + 4));
    out[0] = a.x; out[1] = a.y; out[2] = a.z; out[3] = a.w; out[4] = b.x; out[5] = b.y; out[6] = b.z; out[7] = b.w;
  }
  static __device__ __forceinline__ float one(const float* p) { return *p; }
};

template <typename T>
__global__ void __launch_bounds__(256) k_surface_points(const T* __restrict__ tsdf, VolGeom g, float* __restrict__ pts,
                                                        long long* __restrict__ edge, long long cap, unsigned long long* __restrict__ count,
                                                        const unsigned* __restrict__ slot_of, const unsigned* __restrict__ brick_of,
                                                        const unsigned* __restrict__ pool_used, unsigned pool_cap) {
  const float nanv = __int_as_float(0x7fc00000);
  // dense: every brick of the grid; sparse (slot_of != NULL): the allocated slots -- row r is row r & 63 of slot r >> 6,
  // which holds logical brick brick_of[r >> 6]; a neighbour row in a brick without a slot is unobserved
  const size_t nrows = slot_of ? (size_t)min(*pool_used, pool_cap) * 64 : (size_t)g.bdims[0] * g.bdims[1] * g.bdims[2] * 64;
  auto row_at = [&](int x, int y, int z, bool& ok) -> size_t {       // storage offset of voxel (x, y, z), x a multiple of 8 or any
    if (!slot_of) { ok = true; return (size_t)rf_brick_offset(x, y, z, g.bdims[0], g.bdims[1]); }
    const unsigned sl = slot_of[rf_brick_index(x, y, z, g.bdims[0], g.bdims[1])];
    ok = sl != RF_NO_SLOT;
    return (size_t)sl * RF_BRICK_VOX + rf_in_brick(x, y, z);
  };
  for (size_t row = (size_t)blockIdx.x * blockDim.x + threadIdx.x; row < (nrows + 31) / 32 * 32; row += (size_t)gridDim.x * blockDim.x) {
    float a[8], by[8], bz[8];
    float ax = nanv;
    int i0 = 0, j = 0, k = 0;
    bool live = row < nrows;
    if (live) {
      const size_t b = slot_of ? (size_t)brick_of[row >> 6] : row >> 6;
      const int t = (int)(row & 63), ly = t & 7, lz = t >> 3;
      const int bx = (int)(b % g.bdims[0]), byi = (int)((b / g.bdims[0]) % g.bdims[1]), bzi = (int)(b / ((size_t)g.bdims[0] * g.bdims[1]));
      i0 = bx * 8; j = byi * 8 + ly; k = bzi * 8 + lz;
      live = j < g.dims[1] && k < g.dims[2];
      if (live) {
        SRow<T>::load(tsdf + row * 8, a);
#pragma unroll
        for (int e = 0; e < 8; ++e) { by[e] = nanv; bz[e] = nanv; }
        bool ok;
        size_t o;
        if (j + 1 < g.dims[1]) { o = row_at(i0, j + 1, k, ok); if (ok) SRow<T>::load(tsdf + o, by); }
        if (k + 1 < g.dims[2]) { o = row_at(i0, j, k + 1, ok); if (ok) SRow<T>::load(tsdf + o, bz); }
        if (i0 + 8 < g.dims[0]) { o = row_at(i0 + 8, j, k, ok); if (ok) ax = SRow<T>::one(tsdf + o); }
      }
    }
    // crossing mask: bit 3 e + d
    unsigned m = 0;
    if (live) {
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        if (i0 + e >= g.dims[0]) break;
        const float pa = a[e];
        if (pa != pa) continue;                                   // unobserved
        const float nb[3] = {e < 7 ? a[e + 1] : ax, by[e], bz[e]};
        const bool inx = i0 + e + 1 < g.dims[0];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
          const float pb = nb[d];
          if (pb == pb && (d != 0 || inx) && ((pa > 0.f) != (pb > 0.f))) m |= 1u << (3 * e + d);
        }
      }
    }
    // warp-aggregated append
    const int cnt = __popc(m);
    int pre = cnt;
    const int lane = threadIdx.x & 31;
    for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, pre, o); if (lane >= o) pre += v; }
    const int total = __shfl_sync(0xffffffffu, pre, 31);
    unsigned long long base = 0;
    if (total) {
      if (lane == 31) base = atomicAdd(count, (unsigned long long)total);
      base = __shfl_sync(0xffffffffu, base, 31);
    }
    long long slot = (long long)base + (pre - cnt);
    while (m) {
      const int bit = __ffs(m) - 1;
      m &= m - 1;
      const int e = bit / 3, d = bit - 3 * e;
      if (slot < cap) {
        const float pa = a[e];
        const float pb = d == 0 ? (e < 7 ? a[e + 1] : ax) : (d == 1 ? by[e] : bz[e]);
        const float t = pa / (pa - pb);
        float c[3] = {g.origin[0] + ((float)(i0 + e) + 0.5f) * g.vs, g.origin[1] + ((float)j + 0.5f) * g.vs, g.origin[2] + ((float)k + 0.5f) * g.vs};
        c[d] = fmaf(t, g.vs, c[d]);
        pts[3 * slot] = c[0]; pts[3 * slot + 1] = c[1]; pts[3 * slot + 2] = c[2];
        if (edge) edge[slot] = 3ll * ((long long)(i0 + e) + (long long)g.dims[0] * ((long long)j + (long long)g.dims[1] * k)) + d;
      }
      ++slot;
    }
  }
}

extern "C" int rf_extract_surface_points(const rf_volume* cv, float* points_out_dev, int64_t* edge_out_dev_or_null, int64_t cap,
                                         int64_t* n_out) {
  RF_ARG(cv && points_out_dev && n_out && cap >= 0, "rf_extract_surface_points: bad argument");
  rf_volume* v = const_cast<rf_volume*>(cv);
  RF_CUDA(cudaMemsetAsync(v->upd_count, 0, sizeof(unsigned long long), v->stream));     // the volume's spare 64-bit counter
  const int grid = 148 * 8;
  if (v->g.dtype == RF_F16_W8)
    k_surface_points<__half><<<grid, 256, 0, v->stream>>>((const __half*)v->tsdf, v->g, points_out_dev, (long long*)edge_out_dev_or_null, cap, v->upd_count,
                                                       v->slot_of, v->brick_of, v->pool_used, v->pool_bricks);
  else
    k_surface_points<float><<<grid, 256, 0, v->stream>>>((const float*)v->tsdf, v->g, points_out_dev, (long long*)edge_out_dev_or_null, cap, v->upd_count,
                                                       v->slot_of, v->brick_of, v->pool_used, v->pool_bricks);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  unsigned long long c = 0;
  RF_CUDA(cudaMemcpyAsync(&c, v->upd_count, sizeof(c), cudaMemcpyDeviceToHost, v->stream));
  RF_CUDA(cudaStreamSynchronize(v->stream));
  *n_out = (int64_t)c;
  return RF_OK;
}

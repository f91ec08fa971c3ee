// rf_atlas.cu -- the gather atlas: a derived copy of the TSDF laid out for the fitness kernel's gathers
// (north_star (1): "bricks laid out for texture-like gathers").
//
// Entry (x,y,z) = the 8 TSDF values of the interpolation cell whose low corner is voxel (x,y,z), in the order
// v000 v100 v010 v110 v001 v101 v011 v111 (x fastest), stored in the volume's own dtype: 16 B per voxel for fp16
// volumes, 32 B for fp32.  Entries follow the volume's 8x8x8 brick order, so an x-row of 8 entries is one
// (two) 128-byte line(s).  Unobserved corners keep their NaN sentinel; corners outside the padded grid are NaN.
// The atlas costs 8x the TSDF's memory (2 GiB at 512^3 fp16): it is allocated only when a fitness evaluation
// first needs it, and kept current by refreshing the bricks an integration touched (plus their -x/-y/-z
// neighbours, whose cells reach into the touched brick).
#include "rf_common.cuh"

// One thread per brick a: a needs a refresh iff any brick of a + {0,1}^3 is dirty.
__global__ void k_atlas_mark(const uint8_t* __restrict__ dirty, int BX, int BY, int BZ, unsigned* __restrict__ list,
                             unsigned* __restrict__ count) {
  const size_t nb = (size_t)BX * BY * BZ;
  const size_t a = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool need = false;
  if (a < nb) {
    const int bx = (int)(a % BX), by = (int)((a / BX) % BY), bz = (int)(a / ((size_t)BX * BY));
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      const int x = bx + (c & 1), y = by + ((c >> 1) & 1), z = bz + (c >> 2);
      if (x < BX && y < BY && z < BZ) need |= dirty[((size_t)z * BY + y) * BX + x] != 0;
    }
  }
  const unsigned ballot = __ballot_sync(0xffffffffu, need);
  if (ballot) {
    const int lane = threadIdx.x & 31, leader = __ffs(ballot) - 1;
    unsigned base = 0;
    if (lane == leader) base = atomicAdd(count, __popc(ballot));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (need) list[base + __popc(ballot & ((1u << lane) - 1))] = (unsigned)a;
  }
}

// Sparse volumes: the same test, one thread per ALLOCATED brick (pool slot) instead of per brick of the logical grid -- a brick
// without a slot has no atlas entries to refresh.
__global__ void k_atlas_mark_sparse(const uint8_t* __restrict__ dirty, int BX, int BY, int BZ, const unsigned* __restrict__ brick_of,
                                    const unsigned* __restrict__ pool_used, unsigned pool_cap, unsigned* __restrict__ list,
                                    unsigned* __restrict__ count) {
  const unsigned nslots = min(*pool_used, pool_cap);
  const unsigned s = blockIdx.x * blockDim.x + threadIdx.x;
  bool need = false;
  unsigned a = 0;
  if (s < nslots) {
    a = brick_of[s];
    const int bx = (int)(a % BX), by = (int)((a / BX) % BY), bz = (int)(a / ((unsigned)BX * BY));
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      const int x = bx + (c & 1), y = by + ((c >> 1) & 1), z = bz + (c >> 2);
      if (x < BX && y < BY && z < BZ) need |= dirty[((size_t)z * BY + y) * BX + x] != 0;
    }
  }
  const unsigned ballot = __ballot_sync(0xffffffffu, need);
  if (ballot) {
    const int lane = threadIdx.x & 31, leader = __ffs(ballot) - 1;
    unsigned base = 0;
    if (lane == leader) base = atomicAdd(count, __popc(ballot));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (need) list[base + __popc(ballot & ((1u << lane) - 1))] = a;
  }
}

template <typename T> struct AtlasEntry;
template <> struct AtlasEntry<__half> {
  static __device__ __forceinline__ void store(void* atlas, size_t idx, const __half* h) {
    uint4 o;
    o.x = __half_as_ushort(h[0]) | ((unsigned)__half_as_ushort(h[1]) << 16);
    o.y = __half_as_ushort(h[2]) | ((unsigned)__half_as_ushort(h[3]) << 16);
    o.z = __half_as_ushort(h[4]) | ((unsigned)__half_as_ushort(h[5]) << 16);
    o.w = __half_as_ushort(h[6]) | ((unsigned)__half_as_ushort(h[7]) << 16);
    reinterpret_cast<uint4*>(atlas)[idx] = o;
  }
  static __device__ __forceinline__ __half nan() { return __ushort_as_half((unsigned short)0x7e00); }
  static __device__ __forceinline__ void load_row(const __half* p, __half* out) {
    const uint4 r = *reinterpret_cast<const uint4*>(p);
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const unsigned w = (&r.x)[e];
      out[2 * e] = __ushort_as_half((unsigned short)(w & 0xffffu)); out[2 * e + 1] = __ushort_as_half((unsigned short)(w >> 16));
    }
  }
};
template <> struct AtlasEntry<float> {
  static __device__ __forceinline__ void store(void* atlas, size_t idx, const float* h) {
    float4* p = reinterpret_cast<float4*>(atlas) + 2 * idx;
    p[0] = make_float4(h[0], h[1], h[2], h[3]);
    p[1] = make_float4(h[4], h[5], h[6], h[7]);
  }
  static __device__ __forceinline__ float nan() { return __int_as_float(0x7fc00000); }
  static __device__ __forceinline__ void load_row(const float* p, float* out) {
    const float4 r0 = *reinterpret_cast<const float4*>(p), r1 = *reinterpret_cast<const float4*>(p + 4);
    out[0] = r0.x; out[1] = r0.y; out[2] = r0.z; out[3] = r0.w; out[4] = r1.x; out[5] = r1.y; out[6] = r1.z; out[7] = r1.w;
  }
};

// Persistent CTAs of 256 threads; one brick per CTA pass; each thread builds the two x-adjacent entries (2t, 2t+1) of
// the brick, so a warp stores 1 KiB of contiguous atlas.  The brick and its +x/+y/+z halo (9x9x9 values) are staged in
// shared memory (row stride 10 so that even x is 4-byte aligned for fp16 pairs): every TSDF value is read from global
// memory once.
#define AT_ROW 10
#define AT_PLANE 90
template <typename T> struct AtlasPair;
template <> struct AtlasPair<__half> {      // values at x, x+1, x+2 of one row: one 32-bit and one 16-bit shared load
  static __device__ __forceinline__ void load3(const __half* row, __half& v0, __half& v1, __half& v2) {
    const unsigned w = *reinterpret_cast<const unsigned*>(row);
    v0 = __ushort_as_half((unsigned short)(w & 0xffffu)); v1 = __ushort_as_half((unsigned short)(w >> 16)); v2 = row[2];
  }
};
template <> struct AtlasPair<float> {
  static __device__ __forceinline__ void load3(const float* row, float& v0, float& v1, float& v2) { v0 = row[0]; v1 = row[1]; v2 = row[2]; }
};

template <typename T>
__global__ void __launch_bounds__(256) k_atlas_build(const T* __restrict__ tsdf, void* __restrict__ atlas, int BX, int BY,
                                                     int BZ, const unsigned* __restrict__ list,
                                                     const unsigned* __restrict__ count, uint8_t* __restrict__ dirty,
                                                     const unsigned* __restrict__ slot_of) {
  __shared__ __align__(16) T sh[9 * AT_PLANE];
  const unsigned n = *count;
  // Software pipeline over this CTA's bricks: the global loads of brick q + gridDim.x are issued before the entries of
  // brick q are built and stored, so a pass does not start with an exposed DRAM round trip.
  // Sparse volumes (slot_of != NULL): brick a is stored in pool slot slot_of[a], its entries go to the same slot of the
  // atlas; a brick without a slot is unobserved (a listed one is skipped: its cells read the canonical entry).
  T rowv[8];                                  // threads 0..63: one x-row of the brick
  T hv[2];                                    // threads 64..255: up to two halo values
  unsigned pa = 0;                            // where brick `a` is stored (CTA-uniform)
  auto fetch = [&](unsigned a) {
    const int bx = (int)(a % BX), by = (int)((a / BX) % BY), bz = (int)(a / ((unsigned)BX * BY));
    pa = slot_of ? slot_of[a] : a;
    if (pa == RF_NO_SLOT) return;
    if (threadIdx.x < 64) {
      // the brick itself: 64 x-rows of 8 values, one (two) 128-bit load(s) per row
      AtlasEntry<T>::load_row(tsdf + (size_t)pa * RF_BRICK_VOX + (size_t)(threadIdx.x << 3), rowv);
    } else {
      // the +x / +y / +z halo: 81 + 72 + 64 = 217 values from up to 7 neighbour bricks, at most two per thread
#pragma unroll
      for (int k2 = 0; k2 < 2; ++k2) {
        const int hidx = (int)threadIdx.x - 64 + 192 * k2;
        hv[k2] = AtlasEntry<T>::nan();
        if (hidx < 217) {
          int lx, ly, lz;
          if (hidx < 81) { lx = 8; ly = hidx % 9; lz = hidx / 9; }
          else if (hidx < 153) { const int k = hidx - 81; ly = 8; lx = k & 7; lz = k >> 3; }
          else { const int k = hidx - 153; lz = 8; lx = k & 7; ly = k >> 3; }
          const int cbx = bx + (lx >> 3), cby = by + (ly >> 3), cbz = bz + (lz >> 3);
          if (cbx < BX && cby < BY && cbz < BZ) {
            size_t nb = ((size_t)cbz * BY + cby) * BX + cbx;
            if (slot_of) nb = slot_of[nb];
            if (nb != RF_NO_SLOT) hv[k2] = tsdf[nb * RF_BRICK_VOX + (size_t)(((lz & 7) << 6) | ((ly & 7) << 3) | (lx & 7))];
          }
        }
      }
    }
  };
  unsigned q = blockIdx.x;
  unsigned a = q < n ? list[q] : 0u;
  if (q < n) fetch(a);
  for (; q < n; q += gridDim.x) {
    if (threadIdx.x == 0) dirty[a] = 0;        // every dirty brick is on the list (a brick is its own neighbour 0)
    const unsigned pa_cur = pa;
    if (pa_cur == RF_NO_SLOT) {                // CTA-uniform: nothing stored, nothing to build
      if (q + gridDim.x < n) { a = list[q + gridDim.x]; fetch(a); }
      continue;
    }
    __syncthreads();                           // the previous brick's entries have been read out of sh[]
    if (threadIdx.x < 64) {
      const int ly = threadIdx.x & 7, lz = threadIdx.x >> 3;
#pragma unroll
      for (int e = 0; e < 8; ++e) sh[lz * AT_PLANE + ly * AT_ROW + e] = rowv[e];
    } else {
#pragma unroll
      for (int k2 = 0; k2 < 2; ++k2) {
        const int hidx = (int)threadIdx.x - 64 + 192 * k2;
        if (hidx < 217) {
          int lx, ly, lz;
          if (hidx < 81) { lx = 8; ly = hidx % 9; lz = hidx / 9; }
          else if (hidx < 153) { const int k = hidx - 81; ly = 8; lx = k & 7; lz = k >> 3; }
          else { const int k = hidx - 153; lz = 8; lx = k & 7; ly = k >> 3; }
          sh[lz * AT_PLANE + ly * AT_ROW + lx] = hv[k2];
        }
      }
    }
    __syncthreads();
    if (q + gridDim.x < n) { a = list[q + gridDim.x]; fetch(a); }      // next brick's loads in flight during the build
    {
      const int lx = (threadIdx.x & 3) << 1, ly = (threadIdx.x >> 2) & 7, lz = threadIdx.x >> 5;
      T r[4][3];                                // rows (y,z), (y+1,z), (y,z+1), (y+1,z+1) at x, x+1, x+2
#pragma unroll
      for (int c = 0; c < 4; ++c)
        AtlasPair<T>::load3(&sh[(lz + (c >> 1)) * AT_PLANE + (ly + (c & 1)) * AT_ROW + lx], r[c][0], r[c][1], r[c][2]);
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        T v[8];
#pragma unroll
        for (int c = 0; c < 4; ++c) { v[2 * c] = r[c][e]; v[2 * c + 1] = r[c][e + 1]; }
        AtlasEntry<T>::store(atlas, (size_t)pa_cur * RF_BRICK_VOX + (size_t)((lz << 6) | (ly << 3) | (lx + e)), v);
      }
    }
  }
}

int rf_atlas_sync(rf_volume* v) {
  if (!v->atlas) {
    const size_t esz = v->g.dtype == RF_F16_W8 ? 16 : 32;
    RF_CUDA(cudaMalloc(&v->atlas, (v->nvox + 1) * esz));          // + one canonical all-NaN entry at index nvox
    {
      unsigned canon[8];
      for (int i = 0; i < 8; ++i) canon[i] = v->g.dtype == RF_F16_W8 ? 0x7e007e00u : 0x7fc00000u;
      RF_CUDA(cudaMemcpyAsync((char*)v->atlas + v->nvox * esz, canon, esz, cudaMemcpyHostToDevice, v->stream));
      RF_CUDA(cudaStreamSynchronize(v->stream));                   // canon[] is a stack buffer
    }
    v->graph_valid = 0;
    // every brick is still flagged dirty from create / reset / upload, or the caller integrated before the first
    // evaluation: rebuild everything once.  (Sparse: a brick is flagged when it is allocated and nothing has cleared a
    // flag yet, so the flags already name every allocated brick.)
    if (!v->pool_bricks) RF_CUDA(cudaMemsetAsync(v->brick_dirty, 1, v->nbricks, v->stream));
    v->atlas_stale = 1;
  }
  if (!v->atlas_stale) return RF_OK;
  const int BX = v->g.bdims[0], BY = v->g.bdims[1], BZ = v->g.bdims[2];
  if (!v->refresh_count_zeroed) RF_CUDA(cudaMemsetAsync(v->refresh_count, 0, sizeof(unsigned), v->stream));
  v->refresh_count_zeroed = 0;
  rf_prof_begin(v, 4);
  if (v->pool_bricks)
    k_atlas_mark_sparse<<<(v->pool_bricks + 255) / 256, 256, 0, v->stream>>>(v->brick_dirty, BX, BY, BZ, v->brick_of, v->pool_used,
                                                                           v->pool_bricks, v->refresh_list, v->refresh_count);
  else
    k_atlas_mark<<<(unsigned)((v->nbricks + 255) / 256), 256, 0, v->stream>>>(v->brick_dirty, BX, BY, BZ, v->refresh_list,
                                                                            v->refresh_count);
  rf_prof_end(v, 4);
  const int grid = (int)(v->nbricks < (size_t)148 * 8 ? v->nbricks : (size_t)148 * 8);
  rf_prof_begin(v, 2);
  if (v->g.dtype == RF_F16_W8)
    k_atlas_build<__half><<<grid, 256, 0, v->stream>>>((const __half*)v->tsdf, v->atlas, BX, BY, BZ, v->refresh_list, v->refresh_count, v->brick_dirty, v->slot_of);
  else
    k_atlas_build<float><<<grid, 256, 0, v->stream>>>((const float*)v->tsdf, v->atlas, BX, BY, BZ, v->refresh_list, v->refresh_count, v->brick_dirty, v->slot_of);
  rf_prof_end(v, 2);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(2);
  v->atlas_stale = 0;
  return RF_OK;
}

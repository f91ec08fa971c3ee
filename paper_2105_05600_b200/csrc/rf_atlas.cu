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

// Brick a needs a refresh iff any brick of a + {0,1}^3 is dirty.  One warp per x-row of bricks (by, bz), lanes along x: the
// flags of a row are consecutive bytes, and no thread divides (the first version did five 64-bit divisions per brick and ran
// one thread per brick in 1024 small CTAs: 6.8 us for the 262144 bricks of a 512^3 grid).
__global__ void k_atlas_mark(const uint8_t* __restrict__ dirty, int BX, int BY, int BZ, unsigned* __restrict__ list,
                             unsigned* __restrict__ count) {
  const unsigned row = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (row >= (unsigned)BY * (unsigned)BZ) return;
  const unsigned bz = row / (unsigned)BY, by = row - bz * (unsigned)BY;      // warp-uniform
  const bool yin = by + 1 < (unsigned)BY, zin = bz + 1 < (unsigned)BZ;
  const uint8_t* r00 = dirty + (size_t)row * BX;                              // (by, bz)
  const uint8_t* r10 = r00 + BX;                                              // (by + 1, bz)
  const uint8_t* r01 = r00 + (size_t)BY * BX;                                 // (by, bz + 1)
  const uint8_t* r11 = r01 + BX;
  for (unsigned x0 = 0; x0 < (unsigned)BX; x0 += 32) {
    const unsigned bx = x0 + lane;
    bool need = false;
    if (bx < (unsigned)BX) {
      const bool xin = bx + 1 < (unsigned)BX;
      unsigned any = r00[bx];
      if (xin) any |= r00[bx + 1];
      if (yin) { any |= r10[bx]; if (xin) any |= r10[bx + 1]; }
      if (zin) { any |= r01[bx]; if (xin) any |= r01[bx + 1]; if (yin) { any |= r11[bx]; if (xin) any |= r11[bx + 1]; } }
      need = any != 0;
    }
    const unsigned ballot = __ballot_sync(0xffffffffu, need);
    if (ballot) {
      const int leader = __ffs(ballot) - 1;
      unsigned base = 0;
      if ((int)lane == leader) base = atomicAdd(count, __popc(ballot));
      base = __shfl_sync(0xffffffffu, base, leader);
      if (need) list[base + __popc(ballot & ((1u << lane) - 1))] = bx | (by << 10) | (bz << 20);   // packed (bx, by, bz): k_atlas_build wants the coordinates
    }
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
    if (need) list[base + __popc(ballot & ((1u << lane) - 1))] = (a % (unsigned)BX) | (((a / (unsigned)BX) % (unsigned)BY) << 10) | ((a / ((unsigned)BX * BY)) << 20);   // packed (bx, by, bz)
  }
}

// One aligned 256-bit store (sm_100: STG.E.ENL2.256): a thread's two fp16 entries, or one fp32 entry, as ONE full 32-byte sector.
// (Two 128-bit stores per thread made every warp-wide store touch 32 sectors half-way: twice the L2 write transactions.)
__device__ __forceinline__ void rf_store256(void* p, unsigned a, unsigned b, unsigned c, unsigned d, unsigned e, unsigned f, unsigned g, unsigned h) {
  asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(a), "r"(b), "r"(c), "r"(d), "r"(e), "r"(f), "r"(g), "r"(h) : "memory");
}
template <typename T> struct AtlasEntry;
template <> struct AtlasEntry<__half> {
  // entries idx and idx + 1 (idx even): v0 / v1 = their 8 corner values
  static __device__ __forceinline__ void store2(void* atlas, size_t idx, const __half* v0, const __half* v1) {
    unsigned w[8];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      w[i] = __half_as_ushort(v0[2 * i]) | ((unsigned)__half_as_ushort(v0[2 * i + 1]) << 16);
      w[4 + i] = __half_as_ushort(v1[2 * i]) | ((unsigned)__half_as_ushort(v1[2 * i + 1]) << 16);
    }
    rf_store256(reinterpret_cast<uint4*>(atlas) + idx, w[0], w[1], w[2], w[3], w[4], w[5], w[6], w[7]);
  }
  static __device__ __forceinline__ void store(void* atlas, size_t idx, const __half* h) {
    uint4 o;
    o.x = __half_as_ushort(h[0]) | ((unsigned)__half_as_ushort(h[1]) << 16);
    o.y = __half_as_ushort(h[2]) | ((unsigned)__half_as_ushort(h[3]) << 16);
    o.z = __half_as_ushort(h[4]) | ((unsigned)__half_as_ushort(h[5]) << 16);
    o.w = __half_as_ushort(h[6]) | ((unsigned)__half_as_ushort(h[7]) << 16);
    reinterpret_cast<uint4*>(atlas)[idx] = o;
  }
  static __device__ __forceinline__ __half nan() { return __ushort_as_half((unsigned short)0x7e00); }
  // one x-row of 8 values: a 128-bit global load, four 32-bit shared stores (rows start 4-byte aligned: AT_ROW is even)
  struct Row { uint4 r; };
  static __device__ __forceinline__ void load_row(const __half* p, Row& o) { o.r = *reinterpret_cast<const uint4*>(p); }
  static __device__ __forceinline__ void fill_row(__half* sh_row, const Row& o) {
    unsigned* d = reinterpret_cast<unsigned*>(sh_row);
    d[0] = o.r.x; d[1] = o.r.y; d[2] = o.r.z; d[3] = o.r.w;
  }
};
template <> struct AtlasEntry<float> {
  static __device__ __forceinline__ void store2(void* atlas, size_t idx, const float* v0, const float* v1) {
    float* p = reinterpret_cast<float*>(atlas) + 8 * idx;
    rf_store256(p, __float_as_uint(v0[0]), __float_as_uint(v0[1]), __float_as_uint(v0[2]), __float_as_uint(v0[3]), __float_as_uint(v0[4]), __float_as_uint(v0[5]), __float_as_uint(v0[6]), __float_as_uint(v0[7]));
    rf_store256(p + 8, __float_as_uint(v1[0]), __float_as_uint(v1[1]), __float_as_uint(v1[2]), __float_as_uint(v1[3]), __float_as_uint(v1[4]), __float_as_uint(v1[5]), __float_as_uint(v1[6]), __float_as_uint(v1[7]));
  }
  static __device__ __forceinline__ void store(void* atlas, size_t idx, const float* h) {
    float4* p = reinterpret_cast<float4*>(atlas) + 2 * idx;
    p[0] = make_float4(h[0], h[1], h[2], h[3]);
    p[1] = make_float4(h[4], h[5], h[6], h[7]);
  }
  static __device__ __forceinline__ float nan() { return __int_as_float(0x7fc00000); }
  struct Row { float4 a, b; };
  static __device__ __forceinline__ void load_row(const float* p, Row& o) { o.a = *reinterpret_cast<const float4*>(p); o.b = *reinterpret_cast<const float4*>(p + 4); }
  static __device__ __forceinline__ void fill_row(float* sh_row, const Row& o) {          // rows start 8-byte aligned
    float2* d = reinterpret_cast<float2*>(sh_row);
    d[0] = make_float2(o.a.x, o.a.y); d[1] = make_float2(o.a.z, o.a.w); d[2] = make_float2(o.b.x, o.b.y); d[3] = make_float2(o.b.z, o.b.w);
  }
};

// Persistent CTAs of 256 threads; one brick per CTA pass; each thread builds the two x-adjacent entries (2t, 2t+1) of
// the brick, so a warp stores 1 KiB of contiguous atlas.  The brick and its +x/+y/+z halo (9x9x9 values) are staged in
// shared memory (row stride 10 so that even x is 4-byte aligned for fp16 pairs): every TSDF value is read from global
// memory once.  ncu showed the first version of this kernel bound by instruction issue, three quarters of it index
// arithmetic (decoding a thread's halo elements and the brick coordinates, with integer divisions, twice per pass): a
// thread's halo elements are now decoded ONCE, before the loop, into two packed descriptors, and the refresh list carries
// the brick's coordinates (k_atlas_mark has them anyway) instead of its linear index.
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

// A halo element of a thread, decoded once: shared-memory index (10 bits), voxel offset inside the neighbour brick (9 bits),
// which neighbour (3 bits: +x, +y, +z), valid (1 bit).
__device__ __forceinline__ unsigned rf_halo_desc(int hidx) {
  if (hidx >= 217) return 0u;
  int lx, ly, lz;
  if (hidx < 81) { lx = 8; ly = hidx % 9; lz = hidx / 9; }
  else if (hidx < 153) { const int k = hidx - 81; ly = 8; lx = k & 7; lz = k >> 3; }
  else { const int k = hidx - 153; lz = 8; lx = k & 7; ly = k >> 3; }
  const unsigned sm = (unsigned)(lz * AT_PLANE + ly * AT_ROW + lx);
  const unsigned off = (unsigned)(((lz & 7) << 6) | ((ly & 7) << 3) | (lx & 7));
  const unsigned d = (unsigned)(lx >> 3) | ((unsigned)(ly >> 3) << 1) | ((unsigned)(lz >> 3) << 2);
  return sm | (off << 10) | (d << 19) | (1u << 22);
}

#ifndef RF_ATLAS_MINB
#define RF_ATLAS_MINB 8
#endif
template <typename T>
__global__ void __launch_bounds__(256, RF_ATLAS_MINB) k_atlas_build(const T* __restrict__ tsdf, void* __restrict__ atlas, int BX, int BY,
                                                        int BZ, const unsigned* __restrict__ list,
                                                        const unsigned* __restrict__ count, uint8_t* __restrict__ dirty,
                                                        const unsigned* __restrict__ slot_of) {
  __shared__ __align__(16) T sh[9 * AT_PLANE];
  const unsigned n = *count;
  const unsigned BXY = (unsigned)BX * (unsigned)BY;
  // Software pipeline over this CTA's bricks: the global loads of brick q + gridDim.x are issued before the entries of
  // brick q are built and stored, so a pass does not start with an exposed DRAM round trip.
  // Sparse volumes (slot_of != NULL): brick a is stored in pool slot slot_of[a], its entries go to the same slot of the
  // atlas; a brick without a slot is unobserved (a listed one is skipped: its cells read the canonical entry).
  const bool own = threadIdx.x < 64;          // threads 0..63: one x-row of the brick; 64..255: up to two halo values
  const unsigned hd0 = own ? 0u : rf_halo_desc((int)threadIdx.x - 64), hd1 = own ? 0u : rf_halo_desc((int)threadIdx.x - 64 + 192);
  typename AtlasEntry<T>::Row rowv;
  T hv0 = AtlasEntry<T>::nan(), hv1 = AtlasEntry<T>::nan();
  unsigned pa = 0;                            // where the brick is stored (CTA-uniform)
  unsigned a = 0;                             // its linear index
  auto halo = [&](unsigned hd, unsigned xin, unsigned yin, unsigned zin) -> T {
    T v = AtlasEntry<T>::nan();
    const unsigned d = (hd >> 19) & 7u;
    // the neighbour exists iff it lies inside the grid on every axis the element steps over
    if ((hd >> 22) && (!(d & 1u) || xin) && (!(d & 2u) || yin) && (!(d & 4u) || zin)) {
      size_t nb = (size_t)a + (d & 1u) + ((d >> 1) & 1u) * (unsigned)BX + (d >> 2) * BXY;
      if (slot_of) nb = slot_of[nb];
      if (nb != RF_NO_SLOT) v = tsdf[nb * RF_BRICK_VOX + ((hd >> 10) & 511u)];
    }
    return v;
  };
  auto fetch = [&](unsigned packed) {
    const unsigned bx = packed & 1023u, by = (packed >> 10) & 1023u, bz = packed >> 20;
    a = (bz * (unsigned)BY + by) * (unsigned)BX + bx;
    pa = slot_of ? slot_of[a] : a;
    if (pa == RF_NO_SLOT) return;
    if (own) AtlasEntry<T>::load_row(tsdf + (size_t)pa * RF_BRICK_VOX + (size_t)(threadIdx.x << 3), rowv);
    else {
      const unsigned xin = bx + 1 < (unsigned)BX, yin = by + 1 < (unsigned)BY, zin = bz + 1 < (unsigned)BZ;
      hv0 = halo(hd0, xin, yin, zin);
      hv1 = halo(hd1, xin, yin, zin);
    }
  };
  // this thread's two entries: their rows in shared memory and their place in the brick
  const int elx = (threadIdx.x & 3) << 1, ely = (threadIdx.x >> 2) & 7, elz = threadIdx.x >> 5;
  const T* const erow = &sh[elz * AT_PLANE + ely * AT_ROW + elx];
  const unsigned eoff = (unsigned)((elz << 6) | (ely << 3) | elx);
  T* const own_row = &sh[(threadIdx.x >> 3) * AT_PLANE + (threadIdx.x & 7) * AT_ROW];       // threads 0..63 only
  unsigned q = blockIdx.x;
  if (q < n) fetch(list[q]);
  for (; q < n; q += gridDim.x) {
    if (threadIdx.x == 0) dirty[a] = 0;        // every dirty brick is on the list (a brick is its own neighbour 0)
    const unsigned pa_cur = pa;
    if (pa_cur == RF_NO_SLOT) {                // CTA-uniform: nothing stored, nothing to build
      if (q + gridDim.x < n) fetch(list[q + gridDim.x]);
      continue;
    }
    __syncthreads();                           // the previous brick's entries have been read out of sh[]
    if (own) AtlasEntry<T>::fill_row(own_row, rowv);
    else {
      if (hd0 >> 22) sh[hd0 & 1023u] = hv0;
      if (hd1 >> 22) sh[hd1 & 1023u] = hv1;
    }
    __syncthreads();
    if (q + gridDim.x < n) fetch(list[q + gridDim.x]);                 // next brick's loads in flight during the build
    {
      T r[4][3];                                // rows (y,z), (y+1,z), (y,z+1), (y+1,z+1) at x, x+1, x+2
#pragma unroll
      for (int c = 0; c < 4; ++c)
        AtlasPair<T>::load3(erow + (c >> 1) * AT_PLANE + (c & 1) * AT_ROW, r[c][0], r[c][1], r[c][2]);
      T v0[8], v1[8];
#pragma unroll
      for (int c = 0; c < 4; ++c) { v0[2 * c] = r[c][0]; v0[2 * c + 1] = r[c][1]; v1[2 * c] = r[c][1]; v1[2 * c + 1] = r[c][2]; }
      AtlasEntry<T>::store2(atlas, (size_t)pa_cur * RF_BRICK_VOX + (size_t)eoff, v0, v1);
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
    k_atlas_mark<<<(unsigned)(((size_t)BY * BZ * 32 + 255) / 256), 256, 0, v->stream>>>(v->brick_dirty, BX, BY, BZ, v->refresh_list,
                                                                                   v->refresh_count);
  rf_prof_end(v, 4);
  #ifndef RF_ATLAS_GRID_MULT
#define RF_ATLAS_GRID_MULT 8
#endif
  const int grid = (int)(v->nbricks < (size_t)148 * RF_ATLAS_GRID_MULT ? v->nbricks : (size_t)148 * RF_ATLAS_GRID_MULT);
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

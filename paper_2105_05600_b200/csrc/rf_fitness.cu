// rf_fitness.cu -- steps a0 (back-projection), a1 (overlap mask, fused), a2 (fitness kernel) and a3 (finalise).
//
// Fitness kernel mapping: one thread = one candidate pose (its 3x4 grid-space transform lives in 12
// registers, built in fp64 from the 6-D particle and the centre pose, rounded once); a CTA of 256 candidates
// walks a chunk of the point set.  Point tiles are brought into shared memory by the TMA (cp.async.bulk +
// mbarrier, double-buffered), masked in place (Eq. 19) and then read by every lane at once: one broadcast
// LDS.128 per point per warp, reused across the warp's 32 particles.  Each trilinear sample is ONE 128-bit
// load from the gather atlas (rf_atlas.cu).  Grid = (candidate blocks) x (point splits): one wave of the 148 SMs
// for the paper's 3-5 M-eval iterations, about six waves of >= 64-point chunks for larger problems; each thread ends with one 64-bit integer atomic (n | S in 2^-24 fixed point): integer addition
// is order-independent, so the result is bit-reproducible and no second-stage reduce is needed.
#include "rf_common.cuh"

// Candidates per CTA and resident CTAs per SM: 256 threads, 3 CTAs (80 / 85 registers for fp16 / fp32 volumes, no spills).
// Measured on B200 (config-3 step with the stop rules / with 20 forced iterations, ms): 8 CTAs of 128 threads at 64 registers
// 0.395 / 0.629; 4 of 256 at 64 registers 0.391 / 0.610 (the block scheduler starts an SM's CTAs one after the other: fewer,
// larger CTAs begin their work sooner); 3 of 256 at 80 registers 0.366 / 0.563 (the one-wave grid shrinks again, the chunks
// grow from ~36 to ~44 points and ptxas no longer spills); 2 of 256 with 6 samples in flight 0.358 / 0.561; 1 of 512 0.360 /
// 0.589; 6 of 128 at 78 registers 0.376 / 0.588.  fp32 volumes (config 2, 20 iterations): 7 CTAs of 128 at 72 registers
// 0.554 ms, 3 of 256 at 85 registers 0.535 ms.
#ifndef EV_THREADS_H
#define EV_THREADS_H 256
#endif
#ifndef EV_THREADS_F
#define EV_THREADS_F 256
#endif
#ifndef EV_MINCTAS_H
#define EV_MINCTAS_H 3
#endif
template <typename T> struct EvThreads;
template <> struct EvThreads<__half> { static constexpr int value = EV_THREADS_H; static constexpr int min_ctas = EV_MINCTAS_H; };
template <> struct EvThreads<float> { static constexpr int value = EV_THREADS_F; static constexpr int min_ctas = 896 / EV_THREADS_F; };
#define EV_TILE 256
#ifndef EV_U
#ifndef EV_U
#define EV_U 4          // samples in flight per thread
#endif
#endif

// ---------------------------------------------------------------- a0: back-projection
__global__ void k_backproject(const float* __restrict__ depth, int w, int h, float fx, float fy, float cx, float cy,
                              int stride, int nu, int nv, float4* __restrict__ pts) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= nu * nv) return;
  const int u = stride / 2 + (m % nu) * stride, v = stride / 2 + (m / nu) * stride;
  const float z = __ldg(depth + (size_t)v * w + u);
  const bool ok = z > 0.f && z < INFINITY;
  const float zz = ok ? z : 0.f;
  pts[m] = make_float4(((float)u - cx) * zz / fx, ((float)v - cy) * zz / fy, zz, ok ? 1.f : 0.f);
}

// The three levels of a tracked frame in one launch (same arithmetic as k_backproject, level chosen per thread).
struct Backproject3 { int stride[3], nu[3], count[3]; float4* pts[3]; };
__global__ void k_backproject3(const float* __restrict__ depth, int w, int h, float fx, float fy, float cx, float cy, Backproject3 b,
                               RfBlock256 blk, unsigned long long* __restrict__ blk_dst) {
  if (blk_dst && blockIdx.x == 0 && threadIdx.x < 32) blk_dst[threadIdx.x] = blk.w[threadIdx.x];     // the frame loop's per-call inputs
  int m = blockIdx.x * blockDim.x + threadIdx.x;
  int l = 0;
  if (m >= b.count[0]) { m -= b.count[0]; l = 1; if (m >= b.count[1]) { m -= b.count[1]; l = 2; if (m >= b.count[2]) return; } }
  const int stride = b.stride[l], nu = b.nu[l];
  const int u = stride / 2 + (m % nu) * stride, v = stride / 2 + (m / nu) * stride;
  const float z = __ldg(depth + (size_t)v * w + u);
  const bool ok = z > 0.f && z < INFINITY;
  const float zz = ok ? z : 0.f;
  b.pts[l][m] = make_float4(((float)u - cx) * zz / fx, ((float)v - cy) * zz / fy, zz, ok ? 1.f : 0.f);
}

static inline int lattice_count(int n, int s) { const int h = s / 2; return n > h ? (n - h + s - 1) / s : 0; }

int rf_launch_backproject3(cudaStream_t st, const float* depth_dev, int w, int h, const float K[4], const int stride[3],
                           float4* const pts[3], int m_out[3], const void* block256, void* block_dst) {
  Backproject3 b;
  int total = 0;
  for (int l = 0; l < 3; ++l) {
    b.stride[l] = stride[l]; b.nu[l] = lattice_count(w, stride[l]);
    b.count[l] = b.nu[l] * lattice_count(h, stride[l]); b.pts[l] = pts[l];
    m_out[l] = b.count[l]; total += b.count[l];
  }
  if (total == 0 && !block_dst) return RF_OK;
  RfBlock256 blk;
  if (block_dst) memcpy(&blk, block256, sizeof(blk)); else memset(&blk, 0, sizeof(blk));
  k_backproject3<<<(max(total, 1) + 255) / 256, 256, 0, st>>>(depth_dev, w, h, K[0], K[1], K[2], K[3], b, blk, (unsigned long long*)block_dst);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  return RF_OK;
}

int rf_launch_backproject(cudaStream_t st, const float* depth_dev, int w, int h, const float K[4], int stride,
                          float4* pts, int* m_out) {
  const int nu = lattice_count(w, stride), nv = lattice_count(h, stride);
  *m_out = nu * nv;
  if (nu * nv == 0) return RF_OK;
  k_backproject<<<(nu * nv + 255) / 256, 256, 0, st>>>(depth_dev, w, h, K[0], K[1], K[2], K[3], stride, nu, nv, pts);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  return RF_OK;
}

extern "C" int rf_backproject(const rf_volume* v, const float* depth_dev, int32_t w, int32_t h, const float K[4],
                              int32_t stride, float* points_out_dev, int32_t* m_out) {
  RF_ARG(v && depth_dev && K && points_out_dev && m_out, "rf_backproject: NULL argument");
  RF_ARG(w > 0 && h > 0 && stride > 0, "rf_backproject: sizes must be positive");
  RF_ARG(((uintptr_t)points_out_dev & 15) == 0, "rf_backproject: points_out_dev must be 16-byte aligned");
  int m = 0;
  int rc = rf_launch_backproject(v->stream, depth_dev, w, h, K, stride, (float4*)points_out_dev, &m);
  *m_out = m;
  return rc;
}


// ---------------------------------------------------------------- a2: fitness kernel
// TMA bulk copy + mbarrier plumbing (PTX; SASS shows UBLKCP / SYNCS).
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* b, int n) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(n));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* b, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, unsigned bytes, unsigned long long* b) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(b))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* b, unsigned phase) {
  asm volatile(
      "{\n.reg .pred p;\nRF_WAIT_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra RF_DONE_%=;\nbra RF_WAIT_%=;\nRF_DONE_%=:\n}" ::"r"(
          smem_u32(b)),
      "r"(phase)
      : "memory");
}

struct EvalParams {
  const void* atlas;
  unsigned canon;         // atlas index of the canonical all-NaN entry (read by every sample that leaves the grid)
  int X, Y, Z;
  unsigned sy, sz;        // brick strides in entries: BX*512, BX*BY*512
  float inv_vs;
  float org[3];
  const float4* pts; int M;
  const float* pst; int N;
  int include_centre;
  const double* pose;     // device: 12 doubles, centre pose s*_{k-1}
  const double* scale;    // device: 6 doubles, axis lengths r_{k-1}
  const double* prev;     // device: 12 doubles, s_*^{t-1} (mask mode 1 only)
  MaskCfg mask;
  const int* done;        // device flag or NULL: non-zero -> nothing to do (early stop inside a frame)
  unsigned long long* acc; int* MO;
  int chunk;              // points per split
  unsigned zero;          // always 0, opaque to the compiler (scheduling device in the sample loop)
  const unsigned* slot_of; // sparse volumes: pool slot of every logical brick (RF_NO_SLOT: not allocated), else NULL
  unsigned BX, BXY;        // sparse volumes: bricks per x-row and per z-plane of the logical grid
};

// Grid-space pose of a candidate: m = [R(q(delta_q)) R_c / vs | (t_c + delta_t - origin)/vs - 1/2]  (A2, A3, O4).
__device__ __forceinline__ void rf_candidate_matrix(const EvalParams& p, const double* pose, const double d[6], float m[12]) {
  const double qx = d[0], qy = d[1], qz = d[2];
  const double qw = sqrt(fmax(0.0, 1.0 - (qx * qx + qy * qy + qz * qz)));
  double Rq[9];
  Rq[0] = 1 - 2 * (qy * qy + qz * qz); Rq[1] = 2 * (qx * qy - qz * qw);     Rq[2] = 2 * (qx * qz + qy * qw);
  Rq[3] = 2 * (qx * qy + qz * qw);     Rq[4] = 1 - 2 * (qx * qx + qz * qz); Rq[5] = 2 * (qy * qz - qx * qw);
  Rq[6] = 2 * (qx * qz - qy * qw);     Rq[7] = 2 * (qy * qz + qx * qw);     Rq[8] = 1 - 2 * (qx * qx + qy * qy);
  const double iv = (double)p.inv_vs;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
#pragma unroll
    for (int j = 0; j < 3; ++j)
      m[4 * i + j] = (float)((Rq[3 * i] * pose[j] + Rq[3 * i + 1] * pose[4 + j] + Rq[3 * i + 2] * pose[8 + j]) * iv);
    m[4 * i + 3] = (float)(((pose[4 * i + 3] + d[3 + i]) - (double)p.org[i]) * iv - 0.5);
  }
}

// The 8 corner values of one atlas entry as floats, order v000 v100 v010 v110 v001 v101 v011 v111.
template <typename T> struct Cell;
template <> struct Cell<__half> {
  uint4 raw;
  __device__ __forceinline__ void load(const void* atlas, unsigned off) { raw = __ldg(reinterpret_cast<const uint4*>(atlas) + off); }
  __device__ __forceinline__ unsigned word() const { return raw.x; }
  __device__ __forceinline__ void tie(unsigned t) { raw.x |= t; }
  __device__ __forceinline__ float get(int c) const {
    const unsigned w = (&raw.x)[c >> 1];
    return __half2float(__ushort_as_half((unsigned short)((c & 1) ? (w >> 16) : (w & 0xffffu))));
  }
};
template <> struct Cell<float> {
  float4 lo, hi;
  __device__ __forceinline__ void load(const void* atlas, unsigned off) {
    // one 256-bit load (sm_100: LDG.E.ENL2.256) of the 32-byte-aligned entry
    const float* p = reinterpret_cast<const float*>(atlas) + 8 * (size_t)off;
    asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
        : "=f"(lo.x), "=f"(lo.y), "=f"(lo.z), "=f"(lo.w), "=f"(hi.x), "=f"(hi.y), "=f"(hi.z), "=f"(hi.w)
        : "l"(p));
  }
  __device__ __forceinline__ float get(int c) const { return c < 4 ? (&lo.x)[c] : (&hi.x)[c - 4]; }
  __device__ __forceinline__ unsigned word() const { return __float_as_uint(lo.x); }
  __device__ __forceinline__ void tie(unsigned t) { lo.x = __uint_as_float(__float_as_uint(lo.x) | t); }
};

// One trilinear sample of psi^2 at grid-space point g = m * x.  floor() is taken with the round-down add of
// 1.5*2^23 (exact for |g| < 2^22; anything else, NaN included, lands outside [0, dim-1) and is rejected), which
// keeps the F2I/FRND conversion pipe out of the loop.  A masked point carries NaN in x.x.
template <typename T>
struct Sample {
  Cell<T> cell; float fx, fy, fz; unsigned off;
  template <bool SPARSE = false>
  __device__ __forceinline__ void issue(const EvalParams& p, const float* m, const float4 x) { locate<SPARSE>(p, m, x); cell.load(p.atlas, off); }
  template <bool SPARSE = false>
  __device__ __forceinline__ void locate(const EvalParams& p, const float* m, const float4 x) {
    const float gx = fmaf(m[0], x.x, fmaf(m[1], x.y, fmaf(m[2], x.z, m[3])));
    const float gy = fmaf(m[4], x.x, fmaf(m[5], x.y, fmaf(m[6], x.z, m[7])));
    const float gz = fmaf(m[8], x.x, fmaf(m[9], x.y, fmaf(m[10], x.z, m[11])));
    const float tx = __fadd_rd(gx, 12582912.f), ty = __fadd_rd(gy, 12582912.f), tz = __fadd_rd(gz, 12582912.f);
    const int ix = __float_as_int(tx) - 0x4B400000, iy = __float_as_int(ty) - 0x4B400000, iz = __float_as_int(tz) - 0x4B400000;
    // in-bounds iff 0 <= i0 and i0 + 1 <= dim - 1; a point outside reads the all-NaN entry and is rejected in finish()
    const bool ok = ((unsigned)ix < (unsigned)(p.X - 1)) && ((unsigned)iy < (unsigned)(p.Y - 1)) && ((unsigned)iz < (unsigned)(p.Z - 1));
    fx = gx - (tx - 12582912.f); fy = gy - (ty - 12582912.f); fz = gz - (tz - 12582912.f);
    // brick order: x + (x>>3)*504 + y*8 + (y>>3)*(sy-64) + z*64 + (z>>3)*(sz-512)
    if (SPARSE) {
      // one more dependent load: the pool slot of the cell's brick; a brick that was never allocated is unobserved
      const unsigned bl = ok ? (unsigned)(ix >> 3) + (unsigned)(iy >> 3) * p.BX + (unsigned)(iz >> 3) * p.BXY : 0u;
      const unsigned slot = __ldg(p.slot_of + bl);
      const unsigned inb = (unsigned)(ix & 7) | ((unsigned)(iy & 7) << 3) | ((unsigned)(iz & 7) << 6);
      off = (ok && slot != RF_NO_SLOT) ? slot * RF_BRICK_VOX + inb : p.canon;
      return;
    }
    const unsigned o = (unsigned)ix + (unsigned)(ix >> 3) * 504u + (unsigned)iy * 8u + (unsigned)(iy >> 3) * (p.sy - 64u) +
                       (unsigned)iz * 64u + (unsigned)(iz >> 3) * (p.sz - 512u);
    off = ok ? o : p.canon;
  }
  // Two samples at once on packed binary32 pairs (FADD2 / FFMA2: one issue slot for the two samples' operation; every half is
  // the scalar instruction's result, so nothing changes but the instruction count): floor / fraction of the three grid
  // coordinates ...
  template <bool SPARSE = false>
  static __device__ __forceinline__ void issue2(const EvalParams& p, const float* m, const float4 xa, const float4 xb, Sample& A, Sample& B) {
    const float gxa = fmaf(m[0], xa.x, fmaf(m[1], xa.y, fmaf(m[2], xa.z, m[3]))), gxb = fmaf(m[0], xb.x, fmaf(m[1], xb.y, fmaf(m[2], xb.z, m[3])));
    const float gya = fmaf(m[4], xa.x, fmaf(m[5], xa.y, fmaf(m[6], xa.z, m[7]))), gyb = fmaf(m[4], xb.x, fmaf(m[5], xb.y, fmaf(m[6], xb.z, m[7])));
    const float gza = fmaf(m[8], xa.x, fmaf(m[9], xa.y, fmaf(m[10], xa.z, m[11]))), gzb = fmaf(m[8], xb.x, fmaf(m[9], xb.y, fmaf(m[10], xb.z, m[11])));
    const rf_f2 magic = rf_pk(12582912.f, 12582912.f);
    const rf_f2 gx = rf_pk(gxa, gxb), gy = rf_pk(gya, gyb), gz = rf_pk(gza, gzb);
    const rf_f2 tx = rf_add2_rd(gx, magic), ty = rf_add2_rd(gy, magic), tz = rf_add2_rd(gz, magic);
    float txa, txb, tya, tyb, tza, tzb;
    rf_unpk(tx, txa, txb); rf_unpk(ty, tya, tyb); rf_unpk(tz, tza, tzb);
    rf_unpk(rf_sub2(gx, rf_sub2(tx, magic)), A.fx, B.fx);
    rf_unpk(rf_sub2(gy, rf_sub2(ty, magic)), A.fy, B.fy);
    rf_unpk(rf_sub2(gz, rf_sub2(tz, magic)), A.fz, B.fz);
    A.template address<SPARSE>(p, __float_as_int(txa) - 0x4B400000, __float_as_int(tya) - 0x4B400000, __float_as_int(tza) - 0x4B400000);
    B.template address<SPARSE>(p, __float_as_int(txb) - 0x4B400000, __float_as_int(tyb) - 0x4B400000, __float_as_int(tzb) - 0x4B400000);
    A.cell.load(p.atlas, A.off);
    B.cell.load(p.atlas, B.off);
  }
  template <bool SPARSE = false>
  __device__ __forceinline__ void address(const EvalParams& p, int ix, int iy, int iz) {
    // in-bounds iff 0 <= i0 and i0 + 1 <= dim - 1; a point outside reads the all-NaN entry and is rejected in finish()
    const bool ok = ((unsigned)ix < (unsigned)(p.X - 1)) && ((unsigned)iy < (unsigned)(p.Y - 1)) && ((unsigned)iz < (unsigned)(p.Z - 1));
    if (SPARSE) {
      const unsigned bl = ok ? (unsigned)(ix >> 3) + (unsigned)(iy >> 3) * p.BX + (unsigned)(iz >> 3) * p.BXY : 0u;
      const unsigned slot = __ldg(p.slot_of + bl);
      const unsigned inb = (unsigned)(ix & 7) | ((unsigned)(iy & 7) << 3) | ((unsigned)(iz & 7) << 6);
      off = (ok && slot != RF_NO_SLOT) ? slot * RF_BRICK_VOX + inb : p.canon;
      return;
    }
    const unsigned o = (unsigned)ix + (unsigned)(ix >> 3) * 504u + (unsigned)iy * 8u + (unsigned)(iy >> 3) * (p.sy - 64u) +
                       (unsigned)iz * 64u + (unsigned)(iz >> 3) * (p.sz - 512u);
    off = ok ? o : p.canon;
  }
  // ... and the seven lerps of the trilinear blend; the two psi^2 are added to S in sample order, as the scalar code does.
  static __device__ __forceinline__ void finish2(const Sample& A, const Sample& B, float& S, int& n) {
    const rf_f2 v000 = rf_pk(A.cell.get(0), B.cell.get(0)), v100 = rf_pk(A.cell.get(1), B.cell.get(1));
    const rf_f2 v010 = rf_pk(A.cell.get(2), B.cell.get(2)), v110 = rf_pk(A.cell.get(3), B.cell.get(3));
    const rf_f2 v001 = rf_pk(A.cell.get(4), B.cell.get(4)), v101 = rf_pk(A.cell.get(5), B.cell.get(5));
    const rf_f2 v011 = rf_pk(A.cell.get(6), B.cell.get(6)), v111 = rf_pk(A.cell.get(7), B.cell.get(7));
    const rf_f2 fx = rf_pk(A.fx, B.fx), fy = rf_pk(A.fy, B.fy), fz = rf_pk(A.fz, B.fz);
    const rf_f2 a00 = rf_fma2(fx, rf_sub2(v100, v000), v000), a10 = rf_fma2(fx, rf_sub2(v110, v010), v010);
    const rf_f2 a01 = rf_fma2(fx, rf_sub2(v101, v001), v001), a11 = rf_fma2(fx, rf_sub2(v111, v011), v011);
    const rf_f2 b0 = rf_fma2(fy, rf_sub2(a10, a00), a00), b1 = rf_fma2(fy, rf_sub2(a11, a01), a01);
    float psa, psb;
    rf_unpk(rf_fma2(fz, rf_sub2(b1, b0), b0), psa, psb);
    if (psa == psa) { S = fmaf(psa, psa, S); ++n; }           // NaN = some corner unobserved, or the point is outside
    if (psb == psb) { S = fmaf(psb, psb, S); ++n; }
  }
  __device__ __forceinline__ void finish(float& S, int& n) const {
    const float v000 = cell.get(0), v100 = cell.get(1), v010 = cell.get(2), v110 = cell.get(3);
    const float v001 = cell.get(4), v101 = cell.get(5), v011 = cell.get(6), v111 = cell.get(7);
    const float a00 = fmaf(fx, v100 - v000, v000), a10 = fmaf(fx, v110 - v010, v010);
    const float a01 = fmaf(fx, v101 - v001, v001), a11 = fmaf(fx, v111 - v011, v011);
    const float b0 = fmaf(fy, a10 - a00, a00), b1 = fmaf(fy, a11 - a01, a01);
    const float psi = fmaf(fz, b1 - b0, b0);
    if (psi == psi) { S = fmaf(psi, psi, S); ++n; }           // NaN = some corner unobserved, or the point is outside
  }
};

// Grid: x = particle blocks of EV_THREADS (+ one extra column when the centre is a candidate), y = point splits.
// A particle CTA gives each thread one particle and walks the chunk point by point; the centre CTA gives every
// thread the centre pose (delta = 0) and walks the chunk thread-strided.  Column 0 also counts |O_k|.
template <typename T, bool SPARSE = false>
__global__ void __launch_bounds__(EvThreads<T>::value, EvThreads<T>::min_ctas) k_fitness(EvalParams p) {
  constexpr int EV_THREADS = EvThreads<T>::value;
  rf_grid_dep_trigger();
  __shared__ __align__(16) float4 tile[2][EV_TILE + EV_U];
  __shared__ __align__(8) unsigned long long bar[2];
  const int tid = threadIdx.x;
  const bool centre_cta = p.include_centre && blockIdx.x == gridDim.x - 1;
  const int j = blockIdx.x * EV_THREADS + tid;
  const bool active = centre_cta || j < p.N;
  const int ib = blockIdx.y * p.chunk, ie = min(p.M, ib + p.chunk);
  const int ntiles = (ie - ib + EV_TILE - 1) / EV_TILE;
  if (tid == 0) {
    mbar_init(&bar[0], 1); mbar_init(&bar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    for (int t = 0; t < min(2, ntiles); ++t) {
      const int t0 = ib + t * EV_TILE, cnt = min(EV_TILE, ie - t0);
      mbar_expect_tx(&bar[t], cnt * 16);
      tma_load_1d(tile[t], p.pts + t0, cnt * 16, &bar[t]);
    }
  }
  float pj[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};          // the unit-ball particle (input data, independent of the predecessor)
  if (active && !centre_cta) {
    const float* pp = p.pst + 6 * (size_t)j;
#pragma unroll
    for (int a = 0; a < 6; ++a) pj[a] = __ldg(pp + a);
  }
  // ---- everything below reads what the previous kernel of the frame loop wrote (pose, axis lengths, done flag,
  // cleared accumulators)
  rf_grid_dep_wait();
  // the stop flag, the axis lengths and the centre pose in ONE memory round trip (not three dependent ones)
  const int done = p.done ? *p.done : 0;
  double sc[6], Tc[12];
#pragma unroll
  for (int a = 0; a < 6; ++a) sc[a] = p.scale[a];
#pragma unroll
  for (int a = 0; a < 12; ++a) Tc[a] = p.pose[a];
  if (done) {
    if (tid == 0) for (int t = 0; t < min(2, ntiles); ++t) mbar_wait(&bar[t], 0);   // no bulk copy may outlive the CTA
    return;
  }
  // ---- pose in registers: delta = r (.) p, q = (sqrt(1-|dq|^2), dq), R_j = R(q) R_c, t_j = t_c + dt  (A2, A3)
  float m[12];
  {
    double d[6];
#pragma unroll
    for (int a = 0; a < 6; ++a) d[a] = sc[a] * (double)pj[a];
    rf_candidate_matrix(p, Tc, d, m);
  }
  double Sd = 0.0;
  int n = 0;
  __syncthreads();                     // barrier initialisation visible to every waiter
  for (int t = 0; t < ntiles; ++t) {
    const int b = t & 1;
    const int t0 = ib + t * EV_TILE, cnt = min(EV_TILE, ie - t0);
    mbar_wait(&bar[b], (t >> 1) & 1);
    // ---- a1, in place: a point that is invalid or outside O_k (Eq. 19; A9) gets NaN in x.x and is
    // then rejected by the bounds test of every candidate
    int kept = 0;
    for (int i = tid; i < cnt; i += EV_THREADS) {
      const float4 x = tile[b][i];
      bool keep = x.w != 0.f;
      if (keep && p.mask.mode) {
        const double* Tc = p.pose; const double* P = p.prev;
        const double xw0 = Tc[0] * x.x + Tc[1] * x.y + Tc[2] * x.z + Tc[3];
        const double xw1 = Tc[4] * x.x + Tc[5] * x.y + Tc[6] * x.z + Tc[7];
        const double xw2 = Tc[8] * x.x + Tc[9] * x.y + Tc[10] * x.z + Tc[11];
        const double e0 = xw0 - P[3], e1 = xw1 - P[7], e2 = xw2 - P[11];
        const double y0 = P[0] * e0 + P[4] * e1 + P[8] * e2;
        const double y1 = P[1] * e0 + P[5] * e1 + P[9] * e2;
        const double y2 = P[2] * e0 + P[6] * e1 + P[10] * e2;
        keep = false;
        if (y2 > 0.0) {
          const double u = (double)p.mask.fx * y0 / y2 + (double)p.mask.cx, v = (double)p.mask.fy * y1 / y2 + (double)p.mask.cy;
          keep = u >= 0.0 && u < (double)p.mask.w && v >= 0.0 && v < (double)p.mask.h;
        }
      }
      if (keep) ++kept; else tile[b][i].x = __int_as_float(0x7fc00000);
    }
    if (tid < EV_U) tile[b][cnt + tid].x = __int_as_float(0x7fc00000);     // pad to a multiple of EV_U
    if (blockIdx.x == 0) {
      for (int o = 16; o; o >>= 1) kept += __shfl_xor_sync(0xffffffffu, kept, o);
      if ((tid & 31) == 0 && kept) atomicAdd(p.MO, kept);
    }
    __syncthreads();
    if (active) {
      float S = 0.f;                                  // fp32 over one tile only, then fp64 (A19)
      if (!centre_cta) {
        for (int i0 = 0; i0 < cnt; i0 += EV_U) {
          Sample<T> s[EV_U];
#pragma unroll
          for (int u = 0; u < EV_U; u += 2) Sample<T>::template issue2<SPARSE>(p, m, tile[b][i0 + u], tile[b][i0 + u + 1], s[u], s[u + 1]);   // broadcast LDS.128: same point in every lane
          // Keep all EV_U gathers in flight: the first sample's data is made to depend on the other loads through
          // a mask the compiler cannot see is zero.  Without it ptxas sinks every gather next to its first use
          // (it schedules for cache-hit latency) and the loop runs with one gather in flight per warp.
          {
            unsigned t = 0;
#pragma unroll
            for (int u = 1; u < EV_U; ++u) t ^= s[u].cell.word();
            s[0].cell.tie(t & p.zero);
          }
#pragma unroll
          for (int u = 0; u < EV_U; u += 2) Sample<T>::finish2(s[u], s[u + 1], S, n);
        }
      } else {
        for (int i = tid; i < cnt; i += EV_THREADS) {
          Sample<T> s;
          s.template issue<SPARSE>(p, m, tile[b][i]);
          s.finish(S, n);
        }
      }
      Sd += (double)S;
    }
    if (t + 2 < ntiles) {                             // refill this buffer with tile t+2
      __syncthreads();
      if (tid == 0) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        const int t2 = ib + (t + 2) * EV_TILE, c2 = min(EV_TILE, ie - t2);
        mbar_expect_tx(&bar[b], c2 * 16);
        tma_load_1d(tile[b], p.pts + t2, c2 * 16, &bar[b]);
      }
    }
  }
  unsigned long long packed = n > 0 ? (((unsigned long long)n << RF_ACC_S_BITS) | (unsigned long long)(Sd * RF_ACC_S_SCALE)) : 0ull;
  if (!centre_cta) {
    if (active && packed) atomicAdd(p.acc + p.include_centre + j, packed);
  } else {
    for (int o = 16; o; o >>= 1) packed += __shfl_xor_sync(0xffffffffu, packed, o);
    if ((tid & 31) == 0 && packed) atomicAdd(p.acc, packed);
  }
}

int rf_launch_eval(const rf_volume* cv, cudaStream_t st, const float4* pts, int M, const float* pst, int N,
                   int include_centre, const double* pose_dev, const double* scale_dev, const double* prev_pose_dev,
                   const MaskCfg& mask, const int* done_flag, int set, int pdl) {
  rf_volume* v = const_cast<rf_volume*>(cv);
  if (!v->atlas) { rf_set_error("rf_launch_eval: atlas not built"); return RF_ERR_INVALID_ARG; }
  if (M > RF_MAX_POINTS) { rf_set_error("rf_launch_eval: more than 2^20-1 points"); return RF_ERR_INVALID_ARG; }
  if ((size_t)(N + include_centre) > v->acc_cap) { rf_set_error("rf_launch_eval: accumulators not sized"); return RF_ERR_INVALID_ARG; }
  const int EV_THREADS = v->g.dtype == RF_F16_W8 ? EvThreads<__half>::value : EvThreads<float>::value;
  const int pblocks = (N + EV_THREADS - 1) / EV_THREADS;
  const int cblocks = pblocks + (include_centre ? 1 : 0);
  // One wave: 148 SMs x resident CTAs (queried once).  Small problems get chunks of >= 8 points so that every SM
  // has work; large ones get long chunks (several TMA tiles per CTA) and several waves.
  static int occ[2] = {0, 0};
  const int di = v->g.dtype == RF_F16_W8 ? 1 : 0;
  if (!occ[di]) {
    int nb = 0;
    cudaError_t oe = di ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_fitness<__half, false>, EV_THREADS, 0)
                        : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_fitness<float, false>, EV_THREADS, 0);
    occ[di] = (oe == cudaSuccess && nb > 0) ? nb : 4;
  }
  const int target = 148 * occ[di];
  const int waves = 6, minchunk = 64;        // swept on B200 (config-4 grid): 6 waves of >= 64-point chunks
  int chunk;
  const long long ctas_min = (long long)max(pblocks, 1) * ((M + minchunk - 1) / minchunk);
  if (ctas_min >= (long long)waves * target) {
    // enough work for several waves: about `waves` waves of CTAs (dynamic balance through the block scheduler),
    // chunks between minchunk and 2048 points
    const int splits_w = (int)min((long long)(M + minchunk - 1) / minchunk, max(1LL, (long long)waves * target / max(pblocks, 1)));
    chunk = (M + splits_w - 1) / splits_w;
    chunk = min(2048, max(minchunk, (chunk + EV_U - 1) / EV_U * EV_U));
  } else {
    int splits1 = max(1, target / max(pblocks, 1));      // swept on B200: 0.75 / 1.25 / 1.5 / 2 waves, or counting the centre column, all lose 2-10 % of the config-3 step
    chunk = (M + splits1 - 1) / splits1;
    if (chunk > 160) { splits1 = max(1, 2 * target / max(pblocks, 1)); chunk = (M + splits1 - 1) / splits1; }   // a thread walks its chunk serially: past ~160 points two waves of shorter chunks win (config-4 cell 16384 x 1024: 96.7 -> 82.6 us)
    chunk = min(2048, max(8, (chunk + EV_U - 1) / EV_U * EV_U));
  }
  int splits = (M + chunk - 1) / chunk;
  if (splits > 65535) { chunk = ((M + 65534) / 65535 + EV_U - 1) / EV_U * EV_U; splits = (M + chunk - 1) / chunk; }
  EvalParams p;
  p.atlas = v->atlas; p.canon = (unsigned)v->nvox;
  p.X = v->g.dims[0]; p.Y = v->g.dims[1]; p.Z = v->g.dims[2];
  p.sy = (unsigned)v->g.bdims[0] * RF_BRICK_VOX; p.sz = (unsigned)v->g.bdims[0] * (unsigned)v->g.bdims[1] * RF_BRICK_VOX;
  p.inv_vs = v->g.inv_vs;
  for (int a = 0; a < 3; ++a) p.org[a] = v->g.origin[a];
  p.pts = pts; p.M = M; p.pst = pst; p.N = N; p.include_centre = include_centre;
  p.pose = pose_dev; p.scale = scale_dev; p.prev = prev_pose_dev; p.mask = mask; p.done = done_flag;
  p.acc = v->acc[set]; p.MO = v->d_MO + set; p.chunk = chunk; p.zero = 0u;
  p.slot_of = v->slot_of; p.BX = (unsigned)v->g.bdims[0]; p.BXY = (unsigned)v->g.bdims[0] * (unsigned)v->g.bdims[1];
  dim3 grid(cblocks, splits);
  rf_prof_begin(v, 0);
  cudaError_t le;
  if (v->pool_bricks) {
    if (v->g.dtype == RF_F16_W8) le = rf_launch_pdl(k_fitness<__half, true>, grid, dim3(EV_THREADS), st, pdl, p);
    else le = rf_launch_pdl(k_fitness<float, true>, grid, dim3(EV_THREADS), st, pdl, p);
  } else if (v->g.dtype == RF_F16_W8) le = rf_launch_pdl(k_fitness<__half, false>, grid, dim3(EV_THREADS), st, pdl, p);
  else le = rf_launch_pdl(k_fitness<float, false>, grid, dim3(EV_THREADS), st, pdl, p);
  rf_prof_end(v, 0);
  RF_CUDA(le);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  return RF_OK;
}

// ---------------------------------------------------------------- a3: finalise (Eq. 20; A6)
__device__ __forceinline__ double rf_rho(double S, int n, int M_O, int mode) {
  if (M_O <= 0) return 0.0;
  if (mode == 1) return (n <= 0 || 2 * (long long)n < (long long)M_O) ? 0.0 : exp(-S / (double)n);
  if (mode == 2) return exp(-(S + (double)(M_O - n)));      // Eq. (14), "No Normalize" ablation
  return exp(-(S + (double)(M_O - n)) / (double)M_O);       // tau = 1
}

__global__ void k_finalise(const unsigned long long* __restrict__ acc, int total, const int* __restrict__ M_O, int mode,
                           float* __restrict__ fit, int* __restrict__ cnt, float* __restrict__ S_out) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= total) return;
  const unsigned long long a = acc[c];
  const int n = (int)(a >> RF_ACC_S_BITS);
  const double S = (double)(a & ((1ull << RF_ACC_S_BITS) - 1)) * (1.0 / RF_ACC_S_SCALE);
  fit[c] = (float)rf_rho(S, n, *M_O, mode);
  cnt[c] = n;
  if (S_out) S_out[c] = (float)S;
}

struct PoseScale { double pose[12]; double scale[6]; };
__global__ void k_set_pose(PoseScale ps, double* pose, double* scale) {
  if (threadIdx.x < 12) pose[threadIdx.x] = ps.pose[threadIdx.x];
  if (threadIdx.x < 6) scale[threadIdx.x] = ps.scale[threadIdx.x];
}

extern "C" int rf_eval_particles_ex(const rf_volume* cv, const float* points_dev, int32_t M, const float* pst_dev,
                                    int32_t N, const float pose[12], const float scale[6], int32_t mode,
                                    float* fitness_out_dev, int32_t* count_out_dev, float* S_out_dev) {
  RF_ARG(cv && points_dev && pst_dev && pose && scale && fitness_out_dev && count_out_dev, "rf_eval_particles: NULL argument");
  RF_ARG(M > 0 && N > 0, "rf_eval_particles: M and N must be positive");
  RF_ARG(M <= RF_MAX_POINTS, "rf_eval_particles: M must be below 2^20");
  RF_ARG(((uintptr_t)points_dev & 15) == 0, "rf_eval_particles: points_dev must be 16-byte aligned");
  RF_ARG(mode >= 0 && mode <= 2, "rf_eval_particles: mode must be 0, 1 or 2");
  rf_volume* v = const_cast<rf_volume*>(cv);
  int rc = rf_atlas_sync(v);
  if (rc != RF_OK) return rc;
  rc = rf_ensure_acc(v, (size_t)N, v->stream);
  if (rc != RF_OK) return rc;
  PoseScale ps;
  for (int a = 0; a < 12; ++a) ps.pose[a] = pose[a];
  for (int a = 0; a < 6; ++a) ps.scale[a] = scale[a];
  // the tracker state block doubles as the pose / scale slot of a standalone evaluation
  k_set_pose<<<1, 32, 0, v->stream>>>(ps, v->track->T, v->track->r);
  MaskCfg mk; mk.mode = 0; mk.fx = mk.fy = 1.f; mk.cx = mk.cy = 0.f; mk.w = mk.h = 0;
  rc = rf_launch_eval(v, v->stream, (const float4*)points_dev, M, pst_dev, N, 0, v->track->T, v->track->r, nullptr, mk, nullptr, 0, 0);
  if (rc != RF_OK) return rc;
  k_finalise<<<(N + 255) / 256, 256, 0, v->stream>>>(v->acc[0], N, v->d_MO, mode, fitness_out_dev, count_out_dev, S_out_dev);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(2);
  return RF_OK;
}

extern "C" int rf_eval_particles(const rf_volume* v, const float* points_dev, int32_t M, const float* pst_dev, int32_t N,
                                 const float pose[12], const float scale[6], float* fitness_out_dev, int32_t* count_out_dev) {
  return rf_eval_particles_ex(v, points_dev, M, pst_dev, N, pose, scale, 0, fitness_out_dev, count_out_dev, nullptr);
}

// rf_raycast.cu -- read-out of the fused surface by ray casting through the gather atlas (the paper
// shows reconstructions, and names no read-out algorithm: reading R-R1 in DESIGN.md).
//
// Pixel (u,v) marches x(z) = R ((u-cx)/fx, (v-cy)/fy, 1) z + t (Eq. 1) at the depths z_k = k*step,
// k = 1 .. floor(z_max/step).  The surface is the first k whose samples k-1 and k are both valid trilinear samples
// (all 8 corners observed, A8) with psi_{k-1} > 0 >= psi_k; the depth is the zero of the line through them.
// One sample = one atlas entry (one 128-bit / 256-bit load), exactly as in the fitness kernel.
//
// Ray set-up and the hit run in fp64; the march itself steps a 32.32 fixed-point position (exact integer adds), so the
// cell a sample falls in -- an integer decision -- is the cell the fp64 oracle finds unless the sample lies within
// ~1e-6 voxel of a cell face; the blend runs in fp32.
// Only the depths inside the ray's intersection with the grid's bounding box are visited: samples outside are
// invalid by definition, so skipping them cannot change the first crossing.
#include "rf_common.cuh"

struct RayParams {
  const void* atlas;
  int X, Y, Z, BX, BY;
  size_t canon;        // index of the atlas' all-NaN entry: what a sample outside the grid reads
  double go[3];        // camera centre in grid coordinates: (t - origin)/vs - 1/2
  double Rs[9];        // R / vs
  double inv_fx, inv_fy, cx, cy;
  double step;
  int nk, w, h;
  float* depth;
  float* normal;       // [h,w,3] or NULL
  const unsigned* slot_of;   // sparse volumes: pool slot of a logical brick (RF_NO_SLOT: not allocated), else NULL
};

template <typename T> struct RayEntry;
template <> struct RayEntry<__half> {
  typedef uint4 Raw;
  static __device__ __forceinline__ Raw fetch(const void* atlas, size_t idx) { return __ldg(reinterpret_cast<const uint4*>(atlas) + idx); }
  static __device__ __forceinline__ void unpack(const Raw& r, float* v) {
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x)), b = __half22float2(*reinterpret_cast<const __half2*>(&r.y)),
                 c = __half22float2(*reinterpret_cast<const __half2*>(&r.z)), d = __half22float2(*reinterpret_cast<const __half2*>(&r.w));
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y; v[4] = c.x; v[5] = c.y; v[6] = d.x; v[7] = d.y;
  }
};
template <> struct RayEntry<float> {
  struct Raw { float4 a, b; };
  static __device__ __forceinline__ Raw fetch(const void* atlas, size_t idx) {
    Raw r;
    r.a = __ldg(reinterpret_cast<const float4*>(atlas) + 2 * idx);
    r.b = __ldg(reinterpret_cast<const float4*>(atlas) + 2 * idx + 1);
    return r;
  }
  static __device__ __forceinline__ void unpack(const Raw& r, float* v) {
    const float4 a = r.a, b = r.b;
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
  }
};

// Atlas index of the cell with low corner (ix,iy,iz); the all-NaN entry if the cell leaves the grid or `skip` is set.
// SPARSE: one more dependent load, the pool slot of the cell's brick; a brick without a slot is unobserved.
template <bool SPARSE>
__device__ __forceinline__ size_t rc_index(const RayParams& p, int ix, int iy, int iz, bool skip = false) {
  const bool out = skip | ((unsigned)ix > (unsigned)(p.X - 2)) | ((unsigned)iy > (unsigned)(p.Y - 2)) | ((unsigned)iz > (unsigned)(p.Z - 2));
  unsigned b = ((unsigned)(iz >> 3) * (unsigned)p.BY + (unsigned)(iy >> 3)) * (unsigned)p.BX + (unsigned)(ix >> 3);   // < 2^32 bricks
  if (SPARSE) {
    b = __ldg(p.slot_of + (out ? 0u : b));
    if (out || b == RF_NO_SLOT) return p.canon;
  }
  const size_t idx = (size_t)b * RF_BRICK_VOX + (size_t)(unsigned)(((iz & 7) << 6) | ((iy & 7) << 3) | (ix & 7));
  return out ? p.canon : idx;        // a select, not a branch: the march loop stays straight-line
}
// Trilinear blend of one entry at fractions f: NaN if any corner is unobserved (or the entry is the all-NaN one).
template <typename T>
__device__ __forceinline__ float rc_blend(const typename RayEntry<T>::Raw& raw, float fx, float fy, float fz) {
  float v[8];
  RayEntry<T>::unpack(raw, v);
  const float c00 = fmaf(fx, v[1] - v[0], v[0]), c10 = fmaf(fx, v[3] - v[2], v[2]);
  const float c01 = fmaf(fx, v[5] - v[4], v[4]), c11 = fmaf(fx, v[7] - v[6], v[6]);
  const float c0 = fmaf(fy, c10 - c00, c00), c1 = fmaf(fy, c11 - c01, c01);
  return fmaf(fz, c1 - c0, c0);
}

// 128 threads = a 16x8 pixel tile (small CTAs even out the very different ray lengths); a warp covers 8x4 pixels so
// that its rays stay in neighbouring cells.
#define RC_U 4
template <typename T, bool SPARSE>
__global__ void __launch_bounds__(128, 8) k_raycast(const RayParams p) {
  const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
  const int u = blockIdx.x * 16 + (wrp & 1) * 8 + (lane & 7), v = blockIdx.y * 8 + (wrp >> 1) * 4 + (lane >> 3);
  if (u >= p.w || v >= p.h) return;
  const double dx = ((double)u - p.cx) * p.inv_fx, dy = ((double)v - p.cy) * p.inv_fy;
  double gd[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) gd[a] = p.Rs[3 * a] * dx + p.Rs[3 * a + 1] * dy + p.Rs[3 * a + 2];
  // depths at which the ray is inside the box [-1, dim] on every axis (one voxel of slack on both sides)
  double z0 = 0.0, z1 = (double)p.nk * p.step;
  const int dims[3] = {p.X, p.Y, p.Z};
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double lo = -1.0 - p.go[a], hi = (double)dims[a] - p.go[a];
    if (fabs(gd[a]) < 1e-12) {
      if (lo > 0.0 || hi < 0.0) z1 = -1.0;
    } else {
      const double ta = lo / gd[a], tb = hi / gd[a];
      z0 = fmax(z0, fmin(ta, tb));
      z1 = fmin(z1, fmax(ta, tb));
    }
  }
  float zhit = 0.f;
  double zhit_d = 0.0;
  if (z1 >= z0) {
    // z0, z1 lie in [0, nk*step] and nk < 1e7 (checked on the host): the sample numbers fit an int
    int k0 = (int)floor(z0 / p.step) - 1, k1 = (int)ceil(z1 / p.step) + 1;
    if (k0 < 1) k0 = 1;
    if (k1 > p.nk) k1 = p.nk;
    bool prev_ok = false, found = false;
    float prev = 0.f, ph = 0.f, qh = 0.f;
    int kh = 0;
    // The march runs in 32.32 fixed point: G = position of sample k0, D = increment per sample, both rounded once from
    // fp64; sample k0+i sits at G + i*D exactly (integer adds), i.e. within i * 2^-33 voxel of the fp64 position --
    // 1e-6 voxel after 10^4 in-box samples, far inside the 1e-4 voxel the parity tests treat as a tie.  The cell is
    // the high word, the fraction the low word (its top 23 bits, through the [1,2) mantissa trick): no fp64 and no
    // conversion instructions inside the loop.
    long long G[3], D[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      D[a] = __double2ll_rn(p.step * gd[a] * 4294967296.0);
      G[a] = __double2ll_rn(fma((double)k0 * p.step, gd[a], p.go[a]) * 4294967296.0);
    }
    // RC_U samples per pass: their loads are independent, so RC_U gathers are in flight per ray instead of one; the
    // crossing test then walks them in order.
    for (int kb = k0; kb <= k1 && !found; kb += RC_U) {
      typename RayEntry<T>::Raw raw[RC_U];
      float fx[RC_U], fy[RC_U], fz[RC_U];
#pragma unroll
      for (int j = 0; j < RC_U; ++j) {
        fx[j] = __uint_as_float(0x3f800000u | ((unsigned)G[0] >> 9)) - 1.0f;
        fy[j] = __uint_as_float(0x3f800000u | ((unsigned)G[1] >> 9)) - 1.0f;
        fz[j] = __uint_as_float(0x3f800000u | ((unsigned)G[2] >> 9)) - 1.0f;
        const size_t idx = rc_index<SPARSE>(p, (int)(G[0] >> 32), (int)(G[1] >> 32), (int)(G[2] >> 32), kb + j > k1);
        raw[j] = RayEntry<T>::fetch(p.atlas, idx);
        G[0] += D[0]; G[1] += D[1]; G[2] += D[2];
      }
#pragma unroll
      for (int j = 0; j < RC_U; ++j) {
        const float psi = rc_blend<T>(raw[j], fx[j], fy[j], fz[j]);
        const bool ok = psi == psi;
        const bool cross = !found & ok & prev_ok & (prev > 0.f) & (psi <= 0.f);
        kh = cross ? kb + j : kh;
        ph = cross ? prev : ph;
        qh = cross ? psi : qh;
        found |= cross;
        prev_ok = ok;
        prev = psi;
      }
    }
    if (found) {
      zhit_d = (double)(kh - 1) * p.step + p.step * (double)ph / ((double)ph - (double)qh);
      zhit = (float)zhit_d;
    }
  }
  const size_t pix = (size_t)v * p.w + u;
  p.depth[pix] = zhit;
  if (p.normal) {
    // central differences of half-width one voxel along the world axes: the neighbouring cells at the same fractions
    float n[3] = {__int_as_float(0x7fc00000), __int_as_float(0x7fc00000), __int_as_float(0x7fc00000)};
    if (zhit > 0.f) {
      const double hxg = fma(zhit_d, gd[0], p.go[0]), hyg = fma(zhit_d, gd[1], p.go[1]), hzg = fma(zhit_d, gd[2], p.go[2]);
      const double fa = floor(hxg), fb = floor(hyg), fc = floor(hzg);
      const int hx = (int)fa, hy = (int)fb, hz = (int)fc;
      const float hfx = (float)(hxg - fa), hfy = (float)(hyg - fb), hfz = (float)(hzg - fc);
      typename RayEntry<T>::Raw raw[6];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        raw[2 * a] = RayEntry<T>::fetch(p.atlas, rc_index<SPARSE>(p, hx + (a == 0), hy + (a == 1), hz + (a == 2)));
        raw[2 * a + 1] = RayEntry<T>::fetch(p.atlas, rc_index<SPARSE>(p, hx - (a == 0), hy - (a == 1), hz - (a == 2)));
      }
      float gp[3], gm[3];
      bool all = true;
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        gp[a] = rc_blend<T>(raw[2 * a], hfx, hfy, hfz);
        gm[a] = rc_blend<T>(raw[2 * a + 1], hfx, hfy, hfz);
        all = all && gp[a] == gp[a] && gm[a] == gm[a];
      }
      if (all) {
        const float g0 = gp[0] - gm[0], g1 = gp[1] - gm[1], g2 = gp[2] - gm[2];
        const float len = sqrtf(g0 * g0 + g1 * g1 + g2 * g2);
        if (len > 0.f) { n[0] = g0 / len; n[1] = g1 / len; n[2] = g2 / len; }
      }
    }
    p.normal[3 * pix] = n[0]; p.normal[3 * pix + 1] = n[1]; p.normal[3 * pix + 2] = n[2];
  }
}

extern "C" int rf_raycast(rf_volume* vol, const float K[4], int32_t width, int32_t height, const float pose_c2w[12],
                          float step, float z_max, float* depth_out_dev, float* normals_out_dev_or_null) {
  RF_ARG(vol && K && pose_c2w && depth_out_dev, "rf_raycast: null argument");
  RF_ARG(width > 0 && height > 0 && width <= 16384 && height <= 16384, "rf_raycast: image size out of range");
  RF_ARG(step > 0.f && z_max >= 0.f && isfinite(step) && isfinite(z_max), "rf_raycast: step must be > 0 and z_max >= 0");
  RF_ARG(K[0] != 0.f && K[1] != 0.f, "rf_raycast: focal lengths must be non-zero");
  RF_ARG((double)z_max / (double)step < 1e7, "rf_raycast: more than 1e7 samples per ray");
  int rc = rf_atlas_sync(vol);
  if (rc != RF_OK) return rc;
  RayParams p;
  p.atlas = vol->atlas;
  p.canon = vol->nvox;
  p.X = vol->g.dims[0]; p.Y = vol->g.dims[1]; p.Z = vol->g.dims[2];
  p.BX = vol->g.bdims[0]; p.BY = vol->g.bdims[1];
  const double vs = (double)vol->g.vs;
  for (int a = 0; a < 3; ++a) {
    p.go[a] = ((double)pose_c2w[4 * a + 3] - (double)vol->g.origin[a]) / vs - 0.5;
    for (int b = 0; b < 3; ++b) p.Rs[3 * a + b] = (double)pose_c2w[4 * a + b] / vs;
  }
  p.inv_fx = 1.0 / (double)K[0]; p.inv_fy = 1.0 / (double)K[1]; p.cx = (double)K[2]; p.cy = (double)K[3];
  p.step = (double)step;
  p.nk = (int)floor((double)z_max / (double)step);
  if (p.X < 2 || p.Y < 2 || p.Z < 2) p.nk = 0;     // no interpolation cell exists: nothing to hit
  p.w = width; p.h = height;
  p.depth = depth_out_dev; p.normal = normals_out_dev_or_null;
  p.slot_of = vol->slot_of;
  const dim3 grid((unsigned)((width + 15) / 16), (unsigned)((height + 7) / 8));
  if (vol->pool_bricks) {
    if (vol->g.dtype == RF_F16_W8) k_raycast<__half, true><<<grid, 128, 0, vol->stream>>>(p);
    else k_raycast<float, true><<<grid, 128, 0, vol->stream>>>(p);
  } else if (vol->g.dtype == RF_F16_W8) k_raycast<__half, false><<<grid, 128, 0, vol->stream>>>(p);
  else k_raycast<float, false><<<grid, 128, 0, vol->stream>>>(p);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  return RF_OK;
}

// rf_fitness.cu -- steps a0 (back-projection), a2 (fitness kernel) and a3 (finalise).
//
// Fitness kernel mapping: one thread = one candidate pose (its 3x4 grid-space transform lives in 12
// registers, built in fp64 from the 6-D particle and the centre pose, rounded once); a CTA of 128 candidates
// walks a chunk of the point set staged tile by tile in shared memory (every lane reads the same point:
// one broadcast LDS.128 per point per warp).  Grid = (candidate blocks) x (point splits); each thread ends with
// two integer atomics (S in 2^-32 fixed point, n): integer addition is order-independent, so the result is
// bit-reproducible and no second-stage reduce is needed.
#include "rf_common.cuh"

#define EV_THREADS 128
#define EV_TILE 256

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

static inline int lattice_count(int n, int s) { const int h = s / 2; return n > h ? (n - h + s - 1) / s : 0; }

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
struct EvalParams {
  const void* tsdf;
  int X, Y, Z, BX, BY;
  float inv_vs;
  float org[3];
  const float4* pts; int M;
  const float* pst; int N;
  int include_centre;
  const double* pose;    // device: 12 doubles, centre pose
  const double* scale;   // device: 6 doubles
  const int* done;       // device flag or NULL: non-zero -> nothing to do (early stop inside a frame)
  unsigned long long* acc_S; int* acc_n;
  int chunk;             // points per split
};

template <typename T> __device__ __forceinline__ float ld_tsdf(const T* p, unsigned off);
template <> __device__ __forceinline__ float ld_tsdf<float>(const float* p, unsigned off) { return __ldg(p + off); }
template <> __device__ __forceinline__ float ld_tsdf<__half>(const __half* p, unsigned off) {
  return __half2float(__ushort_as_half(__ldg(reinterpret_cast<const unsigned short*>(p) + off)));
}

template <typename T>
__global__ void __launch_bounds__(EV_THREADS) k_fitness(EvalParams p) {
  if (p.done && *p.done) return;
  __shared__ float4 spts[EV_TILE];
  const int total = p.N + p.include_centre;
  const int c = blockIdx.x * EV_THREADS + threadIdx.x;
  const bool active = c < total;
  // ---- pose in registers: delta = r (.) p, q = (sqrt(1-|dq|^2), dq), R_j = R(q) R_c, t_j = t_c + dt  (A2, A3)
  float m[12];
  {
    double d[6] = {0, 0, 0, 0, 0, 0};
    if (active && !(p.include_centre && c == 0)) {
      const float* pp = p.pst + 6 * (size_t)(c - p.include_centre);
#pragma unroll
      for (int a = 0; a < 6; ++a) d[a] = p.scale[a] * (double)__ldg(pp + a);
    }
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
        m[4 * i + j] = (float)((Rq[3 * i] * p.pose[j] + Rq[3 * i + 1] * p.pose[4 + j] + Rq[3 * i + 2] * p.pose[8 + j]) * iv);
      // grid coordinate g = (x^G - origin)/vs - 1/2
      m[4 * i + 3] = (float)(((p.pose[4 * i + 3] + d[3 + i]) - (double)p.org[i]) * iv - 0.5);
    }
  }
  const T* __restrict__ vol = reinterpret_cast<const T*>(p.tsdf);
  const int i_begin = blockIdx.y * p.chunk;
  const int i_end = min(p.M, i_begin + p.chunk);
  const unsigned sy = (unsigned)p.BX * RF_BRICK_VOX, sz = (unsigned)p.BX * (unsigned)p.BY * RF_BRICK_VOX;
  float S = 0.f;
  int n = 0;
  for (int t0 = i_begin; t0 < i_end; t0 += EV_TILE) {
    const int cnt = min(EV_TILE, i_end - t0);
    __syncthreads();
    for (int i = threadIdx.x; i < cnt; i += EV_THREADS) spts[i] = __ldg(p.pts + t0 + i);
    __syncthreads();
    if (!active) continue;
#pragma unroll 2
    for (int i = 0; i < cnt; ++i) {
      const float4 x = spts[i];
      if (x.w == 0.f) continue;                       // warp-uniform: every lane sees the same point
      const float gx = fmaf(m[0], x.x, fmaf(m[1], x.y, fmaf(m[2], x.z, m[3])));
      const float gy = fmaf(m[4], x.x, fmaf(m[5], x.y, fmaf(m[6], x.z, m[7])));
      const float gz = fmaf(m[8], x.x, fmaf(m[9], x.y, fmaf(m[10], x.z, m[11])));
      const float flx = floorf(gx), fly = floorf(gy), flz = floorf(gz);
      const int ix = (int)flx, iy = (int)fly, iz = (int)flz;
      // in-bounds iff 0 <= i0 and i0 + 1 <= dim - 1
      if ((unsigned)ix < (unsigned)(p.X - 1) && (unsigned)iy < (unsigned)(p.Y - 1) && (unsigned)iz < (unsigned)(p.Z - 1)) {
        const float fx = gx - flx, fy = gy - fly, fz = gz - flz;
        const unsigned ox = ((unsigned)(ix >> 3) << 9) + (unsigned)(ix & 7);
        const unsigned oy = (unsigned)(iy >> 3) * sy + ((unsigned)(iy & 7) << 3);
        const unsigned oz = (unsigned)(iz >> 3) * sz + ((unsigned)(iz & 7) << 6);
        const unsigned dx = (ix & 7) == 7 ? (RF_BRICK_VOX - 7) : 1u;
        const unsigned dy = (iy & 7) == 7 ? (sy - 56u) : 8u;
        const unsigned dz = (iz & 7) == 7 ? (sz - 448u) : 64u;
        const unsigned b000 = ox + oy + oz;
        const float v000 = ld_tsdf<T>(vol, b000), v100 = ld_tsdf<T>(vol, b000 + dx);
        const float v010 = ld_tsdf<T>(vol, b000 + dy), v110 = ld_tsdf<T>(vol, b000 + dy + dx);
        const float v001 = ld_tsdf<T>(vol, b000 + dz), v101 = ld_tsdf<T>(vol, b000 + dz + dx);
        const float v011 = ld_tsdf<T>(vol, b000 + dz + dy), v111 = ld_tsdf<T>(vol, b000 + dz + dy + dx);
        const float a00 = fmaf(fx, v100 - v000, v000), a10 = fmaf(fx, v110 - v010, v010);
        const float a01 = fmaf(fx, v101 - v001, v001), a11 = fmaf(fx, v111 - v011, v011);
        const float b0 = fmaf(fy, a10 - a00, a00), b1 = fmaf(fy, a11 - a01, a01);
        const float psi = fmaf(fz, b1 - b0, b0);
        if (psi == psi) { S = fmaf(psi, psi, S); ++n; }     // NaN = some corner unobserved
      }
    }
  }
  if (active && n > 0) {
    atomicAdd(p.acc_S + c, (unsigned long long)((double)S * RF_S_SCALE));
    atomicAdd(p.acc_n + c, n);
  }
}

int rf_launch_eval(const rf_volume* cv, const float4* pts, int M, const float* pst, int N, int include_centre,
                   const double* pose_dev, const double* scale_dev, const int* done_flag) {
  rf_volume* v = const_cast<rf_volume*>(cv);
  const int total = N + include_centre;
  const int cblocks = (total + EV_THREADS - 1) / EV_THREADS;
  // enough CTAs to fill 148 SMs several times over, but never tiles smaller than 32 points
  int splits = (148 * 12 + cblocks - 1) / cblocks;
  splits = max(1, min(splits, (M + 31) / 32));
  splits = min(splits, 65535);
  int chunk = (M + splits - 1) / splits;
  chunk = (chunk + 31) / 32 * 32;
  splits = max(1, (M + chunk - 1) / chunk);
  if ((size_t)total > v->acc_cap) { rf_set_error("rf_launch_eval: accumulators not sized"); return RF_ERR_INVALID_ARG; }
  EvalParams p;
  p.tsdf = v->tsdf;
  p.X = v->g.dims[0]; p.Y = v->g.dims[1]; p.Z = v->g.dims[2]; p.BX = v->g.bdims[0]; p.BY = v->g.bdims[1];
  p.inv_vs = v->g.inv_vs;
  for (int a = 0; a < 3; ++a) p.org[a] = v->g.origin[a];
  p.pts = pts; p.M = M; p.pst = pst; p.N = N; p.include_centre = include_centre;
  p.pose = pose_dev; p.scale = scale_dev; p.done = done_flag;
  p.acc_S = v->acc_S; p.acc_n = v->acc_n; p.chunk = chunk;
  dim3 grid(cblocks, splits);
  rf_prof_begin(v, 0);
  if (v->g.dtype == RF_F16_W8) k_fitness<__half><<<grid, EV_THREADS, 0, v->stream>>>(p);
  else k_fitness<float><<<grid, EV_THREADS, 0, v->stream>>>(p);
  rf_prof_end(v, 0);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  return RF_OK;
}

// ---------------------------------------------------------------- a3: finalise (Eq. 20; A6)
__global__ void k_count_mask(const float4* __restrict__ pts, int M, int* __restrict__ out) {
  // single CTA, deterministic
  __shared__ int red[32];
  int c = 0;
  for (int i = threadIdx.x; i < M; i += blockDim.x) c += pts[i].w != 0.f;
  for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = c;
  __syncthreads();
  if (threadIdx.x < 32) {
    c = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0;
    for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (threadIdx.x == 0) *out = c;
  }
}

__device__ __forceinline__ double rf_rho(double S, int n, int M_O, int mode) {
  if (M_O <= 0) return 0.0;
  if (mode == 1) return (n <= 0 || 2 * (long long)n < (long long)M_O) ? 0.0 : exp(-S / (double)n);
  return exp(-(S + (double)(M_O - n)) / (double)M_O);       // tau = 1
}

__global__ void k_finalise(unsigned long long* __restrict__ acc_S, int* __restrict__ acc_n, int total,
                           const int* __restrict__ M_O, int mode, float* __restrict__ fit, int* __restrict__ cnt,
                           float* __restrict__ S_out) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= total) return;
  const double S = (double)acc_S[c] * (1.0 / RF_S_SCALE);
  const int n = acc_n[c];
  acc_S[c] = 0; acc_n[c] = 0;                            // read and clear
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
  RF_ARG(((uintptr_t)points_dev & 15) == 0, "rf_eval_particles: points_dev must be 16-byte aligned");
  RF_ARG(mode == 0 || mode == 1, "rf_eval_particles: mode must be 0 or 1");
  rf_volume* v = const_cast<rf_volume*>(cv);
  { int rc0 = rf_ensure_acc(v, (size_t)N); if (rc0 != RF_OK) return rc0; }
  PoseScale ps;
  for (int a = 0; a < 12; ++a) ps.pose[a] = pose[a];
  for (int a = 0; a < 6; ++a) ps.scale[a] = scale[a];
  // the tracker state block doubles as the pose / scale slot of a standalone evaluation
  k_set_pose<<<1, 32, 0, v->stream>>>(ps, v->track->T, v->track->r);
  k_count_mask<<<1, 1024, 0, v->stream>>>((const float4*)points_dev, M, v->d_MO);
  int rc = rf_launch_eval(v, (const float4*)points_dev, M, pst_dev, N, 0, v->track->T, v->track->r, nullptr);
  if (rc != RF_OK) return rc;
  k_finalise<<<(N + 255) / 256, 256, 0, v->stream>>>(v->acc_S, v->acc_n, N, v->d_MO, mode, fitness_out_dev,
                                                    count_out_dev, S_out_dev);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(3);
  return RF_OK;
}

extern "C" int rf_eval_particles(const rf_volume* v, const float* points_dev, int32_t M, const float* pst_dev, int32_t N,
                                 const float pose[12], const float scale[6], float* fitness_out_dev, int32_t* count_out_dev) {
  return rf_eval_particles_ex(v, points_dev, M, pst_dev, N, pose, scale, 0, fitness_out_dev, count_out_dev, nullptr);
}

// rf_common.cuh -- shared declarations of the CUDA path (sm_100a).  Not shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <math.h>
#include <string>

#include "../../include/rosefusion_b200.h"

// ------------------------------------------------------------------------------------------------
// Data layout in HBM.
// The volume is stored as 8x8x8 bricks.  Brick b = ((z>>3)*BY + (y>>3))*BX + (x>>3); inside a brick
// the voxel is at ((z&7)<<6) | ((y&7)<<3) | (x&7).  A brick is 512 voxels: 1 KiB of fp16 TSDF (8 cache
// lines) or 2 KiB of fp32, plus 512 B of u8 weights in a second array with the same indexing (SoA).
// An x-row of 8 voxels is one aligned 128-bit (fp16) / 2x128-bit (fp32) access; 32 lanes cover 4 z-slices
// = 512 contiguous bytes.  Unobserved voxels (W = 0) hold a quiet NaN in the TSDF array so that the
// fitness kernel needs no weight gathers: NaN propagates through the trilinear blend.
// ------------------------------------------------------------------------------------------------
#define RF_BRICK 8
#define RF_BRICK_VOX 512

#define RF_MAX_ITERS 64

struct VolGeom {
  int dims[3];   // logical
  int bdims[3];  // bricks per axis
  float vs, trunc, inv_vs;
  float origin[3];
  int dtype;
  int w_max;
};

// Device-resident tracker state (one per volume).  Doubles: the pose algebra of the swarm update runs in
// fp64 (paper: Kahan sums on the CPU side; here fp64 accumulation, A19).
struct TrackDev {
  double T[12];      // current centre s*_{k-1}
  double Tprev[12];  // s_*^{t-1}
  double r[6];       // axis lengths r_{k-1}
  double r1[6];      // r_1 of this frame
  double final_rho;
  long long evals;
  int empty_run, done, iters_run, status, final_count, argmax;
  int M_O;           // |O_k| of the level about to be evaluated
  int pad;
};

struct rf_volume {
  VolGeom g;
  cudaStream_t stream;
  void* tsdf;        // bricked, __half or float
  uint8_t* weight;   // bricked
  size_t nvox;       // padded voxel count
  size_t nbricks;
  // integration scratch
  float* depth_stage; size_t depth_cap;      // device copy of a host frame
  float* tile_max; size_t tile_cap;          // per 16x16 depth tile: max valid depth
  unsigned* brick_list;                      // active bricks of the current frame
  unsigned* brick_count;                     // [0] = count
  unsigned long long* upd_count;             // voxels updated by the last frame
  // fitness scratch
  unsigned long long* acc_S; int* acc_n; size_t acc_cap;   // per candidate: sum psi^2 in 2^-32 fixed point, valid count
  double* rho; size_t rho_cap;                   // per candidate fitness (double)
  int* cand_n; size_t cand_cap;                  // per candidate valid count
  int* d_MO;
  // tracker scratch
  TrackDev* track;
  float4* pts_raw[3]; float4* pts_k[3]; size_t pts_cap[3];
  rf_track_trace* trace_dev;
  // pinned host staging for results
  TrackDev* track_host; rf_track_trace* trace_host;
  // optional per-kernel timing (rf_profile_*)
  int prof_on;
  cudaEvent_t* prof_ev[2]; int prof_used[2]; int prof_cap[2];
  double prof_ms[2]; long long prof_launches[2];
};

// measurement hooks
extern long long g_rf_launches;
#define RF_LAUNCHED(n) (g_rf_launches += (n))
void rf_prof_begin(rf_volume* v, int which);
void rf_prof_end(rf_volume* v, int which);
void rf_prof_collect(rf_volume* v);

// ---- error plumbing ----
void rf_set_error(const std::string& s);
int rf_cuda_fail(cudaError_t e, const char* what);
#define RF_CUDA(call)                                         \
  do {                                                        \
    cudaError_t _e = (call);                                  \
    if (_e != cudaSuccess) return rf_cuda_fail(_e, #call);    \
  } while (0)
#define RF_ARG(cond, msg)                                     \
  do {                                                        \
    if (!(cond)) { rf_set_error(msg); return RF_ERR_INVALID_ARG; } \
  } while (0)

int rf_ensure(void** p, size_t* cap, size_t need_bytes);   // grow-only device scratch

// ---- brick addressing (device) ----
__device__ __forceinline__ unsigned rf_brick_offset(int x, int y, int z, int BX, int BY) {
  const unsigned b = ((unsigned)(z >> 3) * (unsigned)BY + (unsigned)(y >> 3)) * (unsigned)BX + (unsigned)(x >> 3);
  return b * RF_BRICK_VOX + (unsigned)(((z & 7) << 6) | ((y & 7) << 3) | (x & 7));
}

// internal launchers shared between translation units
// Fitness accumulators.  Each fitness CTA adds its per-candidate partial with integer atomics (S in 2^-32 fixed
// point): integer addition is order-independent, so results are bit-reproducible without a second-stage reduce.
// Consumers (finalise / swarm update) read and clear, so the arrays are zero between launches.
#define RF_S_SCALE 4294967296.0
int rf_ensure_acc(rf_volume* v, size_t total);
int rf_launch_eval(const rf_volume* vol, const float4* pts, int M, const float* pst, int N, int include_centre,
                   const double* pose_dev, const double* scale_dev, const int* done_flag);

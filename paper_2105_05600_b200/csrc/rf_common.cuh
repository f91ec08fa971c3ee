// rf_common.cuh -- shared declarations of the CUDA path (sm_100a).  Not shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <math.h>
#include <string>
#include <string.h>

#include "../../include/rosefusion_b200.h"

// ------------------------------------------------------------------------------------------------
// Data layout in HBM.
// The volume is stored as 8x8x8 bricks.  Brick b = ((z>>3)*BY + (y>>3))*BX + (x>>3); inside a brick
// the voxel is at ((z&7)<<6) | ((y&7)<<3) | (x&7).  A brick is 512 voxels: 1 KiB of fp16 TSDF (8 cache
// lines) or 2 KiB of fp32, plus 512 B of u8 weights in a second array with the same indexing (SoA).
// An x-row of 8 voxels is one aligned 128-bit (fp16) / 2x128-bit (fp32) access; 32 lanes cover 4 z-slices
// = 512 contiguous bytes.  Unobserved voxels (W = 0) hold a quiet NaN in the TSDF array so that the
// fitness kernel needs no weight gathers: NaN propagates through the trilinear blend.
//
// Gather atlas (derived structure, built lazily at the first fitness evaluation and refreshed brick-wise
// after every integration): one entry per voxel holding its whole 2x2x2 interpolation neighbourhood
// (v000 v100 v010 v110 v001 v101 v011 v111), 16 B for fp16 volumes and 32 B for fp32 volumes, same brick
// order as the volume.  One trilinear sample is then ONE aligned 128-bit load (two for fp32) instead of 8
// scalar gathers: the fitness kernel is bound by L1TEX wavefronts, and this cuts them 8x.
// ------------------------------------------------------------------------------------------------
#define RF_BRICK 8
#define RF_BRICK_VOX 512

#define RF_MAX_ITERS 64
#define RF_PROF_SLOTS 6   // 0 fitness kernel, 1 integration update kernel, 2 atlas build, 3 swarm update, 4 tile-max + cull + atlas mark, 5 back-projection + frame begin

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
  double thresh;     // RF_TRACK_THRESH_EQ21: advantage-set threshold carried to the next iteration (<= 0: none)
  long long evals;
  int empty_run, done, iters_run, status, final_count, argmax;
  int M_O;           // |O_k| of the iteration just evaluated
  int pad;
};

// Per-candidate fitness accumulator: one 64-bit word, n in the top 20 bits, S = sum psi^2 in 2^-24 fixed point in
// the low 44 bits (S <= n < 2^20).  CTAs add their partials with ONE integer atomic; integer addition is
// order-independent, so results are bit-reproducible without a second-stage reduce.
#define RF_ACC_S_BITS 44
#define RF_ACC_S_SCALE 16777216.0
#define RF_MAX_POINTS ((1 << 20) - 1)

#define RF_NO_SLOT 0xffffffffu
struct rf_volume {
  VolGeom g;
  cudaStream_t stream;
  void* tsdf;        // bricked, __half or float
  uint8_t* weight;   // bricked
  size_t nvox;       // voxels stored: padded voxel count of a dense volume, 512 x pool capacity of a sparse one
  size_t nbricks;    // bricks of the (logical) grid
  // sparse mode (rf_volume_opts.pool_bricks > 0): bricks live in a pool and are allocated when an integration first sweeps
  // them (k_cull); a logical brick b is stored in pool slot slot_of[b] (RF_NO_SLOT: not allocated, i.e. all unobserved)
  unsigned pool_bricks;        // capacity in bricks; 0 = dense
  unsigned* slot_of;           // [nbricks]
  unsigned* brick_of;          // [pool_bricks]: the logical brick stored in a slot
  unsigned* pool_used;         // device: [0] slots handed out (may exceed the capacity: the excess was dropped), [1] bricks dropped by the last integration
  unsigned* brick_pslot;       // per listed brick of the current frame: its pool slot (k_cull -> k_update)
  // integration scratch
  float* depth_stage; size_t depth_cap;      // device copy of a host frame
  int staged_w, staged_h;                    // size of the current frame's device copy (0 = none)
  const float* cur_frame;                    // device copy of the last host frame consumed (depth_stage or a prefetch slot)
  // frame prefetch (rf_stage_frame): two slots filled on a copy stream while the previous frame is being tracked
  float* pre_buf[2]; size_t pre_cap[2]; int pre_w[2], pre_h[2];
  cudaEvent_t pre_done[2]; cudaEvent_t pre_gate; cudaStream_t copy_stream;
  int pre_head, pre_count;
  float* depth_clean; size_t clean_cap;      // sanitised frame (valid -> d + mu, invalid -> -inf) gathered by k_update
  float* tile_max; size_t tile_cap;          // per 16x16 depth tile: max valid depth
  const float* tile_ready_src; int tile_ready_w, tile_ready_h;   // k_tile_max already ran on this frame (rf_track_integrate)
  cudaEvent_t track_done;                    // end of the frame loop, when fusion kernels are enqueued behind it
  unsigned* brick_list;                      // active bricks of the current frame
  float4* brick_base;                        // per listed brick: camera-space base position (k_cull -> k_update)
  unsigned* brick_count;                     // [0] = count
  unsigned long long* upd_count;             // voxels updated by the last frame
  // gather atlas (see above)
  void* atlas;                 // nvox entries of 16 B (fp16) / 32 B (fp32); NULL until first needed
  uint8_t* brick_dirty;        // per brick: TSDF changed since the atlas was last refreshed
  unsigned* refresh_list; unsigned* refresh_count;
  int atlas_stale;             // host flag: some brick may be dirty
  int refresh_count_zeroed;    // host flag: the integration just enqueued already zeroed refresh_count
  // fitness scratch: two accumulator sets used alternately by consecutive evaluations (the consumer of set b
  // clears set b^1 for the next evaluation, so no memset sits between the launches of a frame)
  unsigned long long* acc[2]; size_t acc_cap;
  int* d_MO;                   // [2] |O_k| counted by the fitness kernel, same alternation
  // CUDA graph of one frame's PFO loop
  cudaStream_t cap_stream; cudaGraphExec_t graph_exec; unsigned long long graph_sig[16]; int graph_valid; int graph_launches;
  void* init_host; void* init_dev;       // per-call inputs of the frame loop (pinned host block + its device copy)
  // tracker scratch
  TrackDev* track;
  float4* pts_raw[3]; size_t pts_cap[3];
  rf_track_trace* trace_dev;
  // pinned host staging for results
  TrackDev* track_host; rf_track_trace* trace_host;
  void* shard;                              // particle-sharded frame loop state (rf_track.cu)
  void* base_scratch; size_t base_cap;      // baselines (rf_baselines.cu): cumulative weights of a resampling
  // optional per-kernel timing (rf_profile_*)
  int prof_on;
  cudaEvent_t* prof_ev[RF_PROF_SLOTS]; int prof_used[RF_PROF_SLOTS]; int prof_cap[RF_PROF_SLOTS];
  double prof_ms[RF_PROF_SLOTS]; long long prof_launches[RF_PROF_SLOTS];
  float* prof_each[RF_PROF_SLOTS]; int prof_each_n[RF_PROF_SLOTS]; int prof_each_cap[RF_PROF_SLOTS];   // individual launch durations, in order
};

// measurement hooks
// Kernel launch counter (rf_launch_count).  Volumes may be driven from different host threads, so the counter is updated
// atomically; while a thread records the frame loop into a CUDA graph its launches are counted apart (t_rf_captured)
// and credited at every replay instead.
extern long long g_rf_launches;
extern thread_local int t_rf_capturing;
extern thread_local long long t_rf_captured;
#define RF_LAUNCHED(n) do { if (t_rf_capturing) t_rf_captured += (n); else __atomic_fetch_add(&g_rf_launches, (long long)(n), __ATOMIC_RELAXED); } while (0)
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

__device__ __forceinline__ unsigned rf_brick_index(int x, int y, int z, int BX, int BY) {
  return ((unsigned)(z >> 3) * (unsigned)BY + (unsigned)(y >> 3)) * (unsigned)BX + (unsigned)(x >> 3);
}
__device__ __forceinline__ unsigned rf_in_brick(int x, int y, int z) { return (unsigned)(((z & 7) << 6) | ((y & 7) << 3) | (x & 7)); }

// internal launchers shared between translation units
int rf_ensure_acc(rf_volume* v, size_t total, cudaStream_t st);   // sizes and zeroes both accumulator sets
// 256 bytes of per-call input that ride along as kernel arguments of a launch the call makes anyway (k_backproject3) and are
// dropped into device memory by its first warp: the frame loop's first kernel then reads them from L2 instead of fetching a
// pinned host block over PCIe (~2 us on the frame's critical path).
struct RfBlock256 { unsigned long long w[32]; };
int rf_integrate_prelaunch(rf_volume* v, const float* d_dev, int w, int h);   // the pose-independent first kernel of a fusion
int rf_atlas_sync(rf_volume* v);                                   // allocate / refresh the gather atlas (stream-ordered)
struct MaskCfg { int mode; float fx, fy, cx, cy; int w, h; };      // mode 0: keep every valid point; 1: Eq. 19 overlap test
int rf_launch_eval(const rf_volume* vol, cudaStream_t st, const float4* pts, int M, const float* pst, int N,
                   int include_centre, const double* pose_dev, const double* scale_dev, const double* prev_pose_dev,
                   const MaskCfg& mask, const int* done_flag, int set, int pdl);

// Packed binary32 pairs (sm_100 FFMA2 / FADD2): two IEEE operations per issue slot, each half rounded exactly like the scalar
// instruction (so packing changes no result bit).
typedef unsigned long long rf_f2;
__device__ __forceinline__ rf_f2 rf_pk(float lo, float hi) { rf_f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void rf_unpk(rf_f2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ rf_f2 rf_c2(const float2& c) { return *reinterpret_cast<const rf_f2*>(&c); }
__device__ __forceinline__ rf_f2 rf_fma2(rf_f2 a, rf_f2 b, rf_f2 c) { rf_f2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ rf_f2 rf_add2(rf_f2 a, rf_f2 b) { rf_f2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ rf_f2 rf_add2_rd(rf_f2 a, rf_f2 b) { rf_f2 r; asm("add.rm.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ rf_f2 rf_sub2(rf_f2 a, rf_f2 b) { rf_f2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }

// Programmatic dependent launch (PDL): a kernel launched with rf_launch_pdl may start while its predecessor in
// the stream is still draining; it runs its independent prologue and then blocks in rf_grid_dep_wait() until the
// predecessor has completed and its writes are visible.  rf_grid_dep_trigger() in the predecessor allows that
// early start.  Both are no-ops for ordinary launches.
__device__ __forceinline__ void rf_grid_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void rf_grid_dep_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <typename... KArgs, typename... Args>
inline cudaError_t rf_launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, cudaStream_t st, int pdl, Args... args) {
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = 0; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, args...);
}

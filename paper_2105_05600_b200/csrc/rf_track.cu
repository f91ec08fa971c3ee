// rf_track.cu -- steps a3 (finalise), a4 (swarm update), a5 (iteration control): Algorithm 1 with the
// whole loop on the device.  The paper runs the update on the CPU with one CPU<->GPU round trip per iteration
// (Fig. 8); here state (pose, axis lengths, flags) stays in device memory, one frame's loop is a
// CUDA graph of 2 kernels per iteration (k_fitness -> k_swarm_update), and a `done` flag turns the remaining
// launches of a frame into no-ops once a stop rule fires.
#include "rf_common.cuh"
#include <string.h>
#include <stdlib.h>
#include <cooperative_groups.h>
namespace cg = cooperative_groups;

#define UP_THREADS 512
#define UP_NQ 10          // partial sums per CTA: sum w, sum w*rho, sum w*delta[6], |APS|, (unused)

int rf_launch_backproject3(cudaStream_t st, const float* depth_dev, int w, int h, const float K[4], const int stride[3],
                           float4* const pts[3], int m_out[3], const void* block256, void* block_dst);

struct TrackCfg { float fx, fy, cx, cy; int w, h, mode, early_stop, iters, variant; };
struct TrackInit { double T[12]; double Tprev[12]; double r[6]; double thresh; int has_r0; int pad; };
static_assert(sizeof(TrackInit) == sizeof(RfBlock256), "TrackInit travels as an RfBlock256");

// Start of a frame: state from the staged TrackInit, both accumulator sets and both |O_k| counters zeroed.
__global__ void k_track_begin(const TrackInit* __restrict__ in, TrackDev* st, unsigned long long* acc0,
                              unsigned long long* acc1, int clear_n, int* MO) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < clear_n) { acc0[i] = 0ull; acc1[i] = 0ull; }
  if (blockIdx.x != 0) return;
  if (threadIdx.x < 12) { st->T[threadIdx.x] = in->T[threadIdx.x]; st->Tprev[threadIdx.x] = in->Tprev[threadIdx.x]; }
  if (threadIdx.x < 6) { st->r[threadIdx.x] = in->r[threadIdx.x]; st->r1[threadIdx.x] = in->r[threadIdx.x]; }
  if (threadIdx.x == 0) {
    st->final_rho = 0; st->thresh = in->thresh; st->evals = 0; st->empty_run = 0; st->done = 0; st->iters_run = 0; st->status = 0;
    st->final_count = 0; st->argmax = 0; st->M_O = 0;
    MO[0] = 0; MO[1] = 0;
  }
}

__device__ __forceinline__ double rho_of(double S, int n, int M_O, int mode) {
  if (M_O <= 0) return 0.0;
  if (mode == 1) return (n <= 0 || 2 * (long long)n < (long long)M_O) ? 0.0 : exp(-S / (double)n);
  if (mode == 2) return exp(-(S + (double)(M_O - n)));      // Eq. (14): "No Normalize" ablation
  return exp(-(S + (double)(M_O - n)) / (double)M_O);       // Eq. (20), tau = 1 (A6)
}
// rho = exp(-x): the exponent alone orders candidates (monotone), so the update kernel compares exponents and calls
// exp only for candidates that can enter the advantage set.
// inv_MO = 1 / M_O, computed once per thread: a candidate costs a product, not an fp64 division (the fp64 pipe, with
// 16 warps per CTA, is what the per-candidate phase waits on).
__device__ __forceinline__ double x_of(double S, int n, int M_O, double inv_MO, int mode) {
  if (M_O <= 0) return INFINITY;
  if (mode == 1) return (n <= 0 || 2 * (long long)n < (long long)M_O) ? INFINITY : S / (double)n;
  if (mode == 2) return S + (double)(M_O - n);
  return (S + (double)(M_O - n)) * inv_MO;
}
__device__ __forceinline__ double acc_S(unsigned long long a) { return (double)(a & ((1ull << RF_ACC_S_BITS) - 1)) * (1.0 / RF_ACC_S_SCALE); }
__device__ __forceinline__ int acc_n(unsigned long long a) { return (int)(a >> RF_ACC_S_BITS); }

// first tracked frame (A11): r_0,d = 2 (1 - rho(T_0)) / sqrt(6) + eps from the centre alone on level 0.
__global__ void k_init_r0(const unsigned long long* acc, const int* MO, TrackDev* st, TrackCfg cfg) {
  if (threadIdx.x != 0) return;
  const unsigned long long a = acc[0];
  const double rho0 = rho_of(acc_S(a), acc_n(a), *MO, cfg.mode);
  for (int d = 0; d < 6; ++d) st->r[d] = 2.0 * (1.0 - rho0) / sqrt(6.0) + 1e-3;
  st->evals += *MO;
}

// T_out = Delta(delta) o T_in  (MovePST; A2: left-multiplied increment, world-frame translation)
__device__ void apply_delta(const double* Tin, const double* d, double* Tout) {
  const double qx = d[0], qy = d[1], qz = d[2];
  const double qw = sqrt(fmax(0.0, 1.0 - (qx * qx + qy * qy + qz * qz)));
  double Rq[9];
  Rq[0] = 1 - 2 * (qy * qy + qz * qz); Rq[1] = 2 * (qx * qy - qz * qw);     Rq[2] = 2 * (qx * qz + qy * qw);
  Rq[3] = 2 * (qx * qy + qz * qw);     Rq[4] = 1 - 2 * (qx * qx + qz * qz); Rq[5] = 2 * (qy * qz - qx * qw);
  Rq[6] = 2 * (qx * qz - qy * qw);     Rq[7] = 2 * (qy * qz + qx * qw);     Rq[8] = 1 - 2 * (qx * qx + qy * qy);
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) Tout[4 * i + j] = Rq[3 * i] * Tin[j] + Rq[3 * i + 1] * Tin[4 + j] + Rq[3 * i + 2] * Tin[8 + j];
    Tout[4 * i + 3] = Tin[4 * i + 3] + d[3 + i];
  }
}

struct UpdParams {
  const unsigned long long* acc;      // this evaluation's accumulators (candidate 0 = centre)
  unsigned long long* acc_next;       // the other set: cleared here for the next evaluation
  int clear_n;
  const int* MO; int* MO_next;
  int N; const float* pst;
  TrackDev* st; TrackCfg cfg;
  int k, k0, level;
  rf_track_trace* trace;
  // particle-sharded evaluation: this launch sees a slice of the level's template
  int idx_off;          // global index of the slice's first particle (candidate c >= 1 is particle idx_off + c - 1)
  int n_total;          // particles of the whole level (evals bookkeeping)
  double* row_out;      // partial mode: the cluster's folded row goes here (UP_ROW doubles) instead of being applied
};
#define UP_ROW 16         // a rank's row: UP_STRIDE partial results, rho_ref, M_O, pad

#define UP_STRIDE (UP_NQ + 3)

// The serial part of an iteration (one thread): Eq. (15)-(18), (21), the corner cases of P:L292 and the stop rules of
// P:L306, from the folded sums `tot` (sum w, sum w rho, sum w delta[6], |APS|, -, best exponent, best index, its count).
__device__ void swarm_serial_step(const UpdParams& p, const double* tot, const double* Tin, int empty_run_in, double* r,
                                  double rho_ref, int M_O, int total) {
  TrackDev* st = p.st;
  const double sw = tot[0], swr = tot[1];
  const int n_aps = (int)tot[8];
  const int best = (int)tot[UP_NQ + 1];
  double dstar[6] = {0, 0, 0, 0, 0, 0}, rhat[6], rho_tilde = 0, Tn[12];
  int empty_run = empty_run_in, stop = 0;
  if (n_aps > 0) {
    const double inv_sw = 1.0 / sw;                                      // one division, then products (serial thread)
    for (int d = 0; d < 6; ++d) dstar[d] = tot[2 + d] * inv_sw;          // Eq. (15) in the chart at s*_{k-1} (A3)
    rho_tilde = swr * inv_sw;                                            // Eq. (21)
    apply_delta(Tin, dstar, Tn);
    double nv = 0;
    for (int d = 0; d < 6; ++d) nv += dstar[d] * dstar[d];               // v = s_k^* - s_{k-1}^*  (Eq. 16)
    nv = sqrt(nv);
    const double inv_nv = nv > 0 ? 1.0 / nv : 0.0;
    for (int d = 0; d < 6; ++d) {                                        // Eq. (17), A4; ablations of Fig. 11
      const double aniso = fabs(dstar[d]) * inv_nv, iso = 1.0 - rho_tilde;
      if (p.cfg.variant & RF_TRACK_RESCALE_ISO) rhat[d] = iso / sqrt(6.0) + 1e-3;
      else if (p.cfg.variant & RF_TRACK_RESCALE_ANISO) rhat[d] = aniso + 1e-3;
      else rhat[d] = iso * aniso + 1e-3;
    }
    empty_run = 0;
  } else {
    for (int a = 0; a < 12; ++a) Tn[a] = Tin[a];
    for (int d = 0; d < 6; ++d) rhat[d] = 2.0 * (1.0 - rho_ref) / sqrt(6.0) + 1e-3;   // P:L292, A13
    empty_run += 1;
  }
  for (int d = 0; d < 6; ++d) r[d] = 0.1 * r[d] + 0.9 * rhat[d];         // Eq. (18), beta = 0.1
  if (empty_run >= 2) stop = 1;
  else if (n_aps > 0) {
    double mx = 0;
    for (int d = 0; d < 6; ++d) mx = fmax(mx, fabs(dstar[d]));
    if (mx < 1e-6) stop = 2;                                             // P:L306, A16
  }
  for (int a = 0; a < 12; ++a) st->T[a] = Tn[a];
  for (int d = 0; d < 6; ++d) st->r[d] = r[d];
  if (p.k == 1) for (int d = 0; d < 6; ++d) st->r1[d] = r[d];            // P:L286  r_0^{t+1} = r_1^t
  st->empty_run = empty_run;
  st->iters_run = p.k - p.k0;
  st->final_rho = n_aps > 0 ? rho_tilde : rho_ref;
  st->thresh = (p.cfg.variant & RF_TRACK_THRESH_EQ21) ? (n_aps > 0 ? rho_tilde : rho_ref) : 0.0;
  st->final_count = (int)tot[UP_NQ + 2];
  st->argmax = best;
  st->M_O = M_O;
  st->evals += (long long)total * M_O;
  if (M_O == 0) st->status |= RF_TRACK_NO_POINTS;
  if (p.cfg.early_stop && stop) { st->done = 1; st->status |= (stop == 1 ? RF_TRACK_STOP_EMPTY : RF_TRACK_STOP_SMALL); }
  if (p.trace) {
    rf_track_trace& tr = p.trace[p.k - p.k0 - 1];
    tr.level = p.level; tr.M_O = M_O; tr.n_aps = n_aps; tr.argmax = best; tr.stop = stop; tr.empty_run = empty_run;
    tr.rho_ref = rho_ref; tr.rho_max = exp(-tot[UP_NQ]); tr.rho_tilde = rho_tilde; tr.sum_omega = n_aps > 0 ? sw : 0.0;
    for (int d = 0; d < 6; ++d) { tr.delta_star[d] = dstar[d]; tr.r[d] = r[d]; }
    for (int a = 0; a < 12; ++a) tr.pose[a] = Tn[a];
  }
}


// a3 + a4 + a5 for iteration k (1-based).  ONE thread-block cluster of up to 8 CTAs x 512 threads: each thread
// finalises its candidates (Eq. 20) and forms their APS terms in ascending order; fixed-shape warp / CTA reductions
// give one row per CTA, written straight into the shared memory of the cluster's first CTA (distributed shared
// memory); after one cluster barrier that CTA folds the rows in rank order -- the reduction tree depends only on N, so
// results are bit-reproducible -- and one thread applies Eq. 15-18, 21 and the stop rules in fp64 (the paper's
// Kahan-summed CPU step).  No global-memory round trip or ticket sits between the phases.
#define UP_MAX_CLUSTER 8
__global__ void __launch_bounds__(UP_THREADS) k_swarm_update(UpdParams p) {
  cg::cluster_group cluster = cg::this_cluster();
  const unsigned C = cluster.num_blocks(), rank = cluster.block_rank();
  __shared__ double sh[UP_THREADS / 32][UP_STRIDE];
  __shared__ double rows[UP_MAX_CLUSTER][UP_STRIDE];      // used in the first CTA only
  __shared__ double tot[UP_STRIDE];
  TrackDev* st = p.st;
  rf_grid_dep_trigger();
  // every CTA of the cluster announces that it is running; a CTA waits for all of them before its first store into
  // another CTA's shared memory (distributed shared memory may only be accessed once the target block exists)
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  const int total = p.N + 1;
  const int gtid = (int)rank * UP_THREADS + threadIdx.x, gstride = (int)C * UP_THREADS;
  // The candidates of this thread's first pass (for the paper's template sizes: its only pass).  Their particles are inputs,
  // not results of the fitness kernel: they are fetched before the dependency wait, under that kernel's tail ...
  float pj0[3][6];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const int c = gtid + k * gstride;
#pragma unroll
    for (int d = 0; d < 6; ++d) pj0[k][d] = (c > 0 && c < total) ? __ldg(p.pst + 6 * (size_t)(c - 1) + d) : 0.f;
  }
  rf_grid_dep_wait();
  // ... and their accumulators in the same memory round trip as everything else this thread needs from the previous kernels
  // (not in a second one behind the `done` test)
  const int done = st->done;
  const double thresh_in = st->thresh;
  const int M_O = *p.MO;
  const unsigned long long a0 = p.acc[0];
  unsigned long long acc0[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) { const int c = gtid + k * gstride; acc0[k] = c < total ? p.acc[c] : 0ull; }
  double r[6];
#pragma unroll
  for (int d = 0; d < 6; ++d) r[d] = st->r[d];
  // the thread that applies Eq. 15-18 at the end fetches the pose and the empty-run counter in this same round trip
  // (nothing else writes them during this kernel), not in its serial tail
  // (parked in shared memory: no registers held across the kernel)
  __shared__ double Tin[12];
  __shared__ int empty_run_in;
  if (gtid == 0) {
#pragma unroll
    for (int a = 0; a < 12; ++a) Tin[a] = st->T[a];
    empty_run_in = st->empty_run;
  }
  if (done) return;                                       // uniform over the cluster
  for (int i = gtid; i < p.clear_n; i += gstride) p.acc_next[i] = 0ull;
  if (gtid == 0) *p.MO_next = 0;
  const double inv_MO = M_O > 0 ? 1.0 / (double)M_O : 0.0;
  const double x_0 = x_of(acc_S(a0), acc_n(a0), M_O, inv_MO, p.cfg.mode);
  // threshold of the advantage set: the exact fitness of s*_{k-1} on this point set (A14), or, in the Eq. (21) variant,
  // the value carried from the previous iteration (the exponent filter below is then taken a hair wider: membership
  // itself is decided on rho)
  const bool carried = (p.cfg.variant & RF_TRACK_THRESH_EQ21) && thresh_in > 0.0;
  const double rho_ref = carried ? thresh_in : exp(-x_0);
  const double x_ref = carried ? -log(thresh_in) + 1e-9 : x_0;
  // ---- per candidate: rho_c, APS membership (rho > rho_ref), omega = rho - rho_ref, Eq. (15)/(21) terms
  double q[UP_NQ];
#pragma unroll
  for (int i = 0; i < UP_NQ; ++i) q[i] = 0.0;
  double bv = INFINITY; int bi = 0x7fffffff, bn = 0;       // best = smallest exponent x (largest rho), ties -> lowest index
  // three candidates per pass: all their loads (accumulator word + particle) are issued before any of them is used,
  // so a thread pays one memory round trip per pass, not one per candidate; accumulation order stays ascending in c
  for (int c0 = gtid; c0 < total; c0 += 3 * gstride) {
    unsigned long long a[3];
    float pj[3][6];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const int c = c0 + k * gstride;
      if (c0 == gtid) {                                      // first pass: fetched above
        a[k] = acc0[k];
#pragma unroll
        for (int d = 0; d < 6; ++d) pj[k][d] = pj0[k][d];
      } else {
        a[k] = c < total ? p.acc[c] : 0ull;
#pragma unroll
        for (int d = 0; d < 6; ++d) pj[k][d] = (c > 0 && c < total) ? __ldg(p.pst + 6 * (size_t)(c - 1) + d) : 0.f;
      }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const int c = c0 + k * gstride;
      if (c >= total) break;
      const int n = acc_n(a[k]);
      const double xc = c == 0 ? x_0 : x_of(acc_S(a[k]), n, M_O, inv_MO, p.cfg.mode);
      if (xc < bv || bi == 0x7fffffff) { bv = xc; bi = c == 0 ? 0 : c + p.idx_off; bn = n; }   // ascending c: ties keep the lowest index (A18)
      const double rc = (c > 0 && xc < x_ref) ? exp(-xc) : 0.0;      // exp only where membership is possible
      if (rc > rho_ref) {                                            // strict, on rho itself
        const double w = rc - rho_ref;
        q[0] += w; q[1] += w * rc; q[8] += 1.0;
#pragma unroll
        for (int d = 0; d < 6; ++d) q[2 + d] += w * (r[d] * (double)pj[k][d]);
      }
    }
  }
  // warp reduce (sums; argmax with ties -> lowest index, A18).  The sums are reduced transposed: in each of four
  // rounds a lane keeps one half of its quantities and hands the other half to its partner, so 16 slots cost
  // 8 + 4 + 2 + 1 (+ 1 final) exchanges instead of 5 per quantity; lanes 2i and 2i+1 end with the warp total of
  // quantity i.  The shape is fixed, so the result is bit-reproducible.
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double v[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = i < UP_NQ ? q[i] : 0.0;
#pragma unroll
  for (int half = 8, o = 16; half >= 1; half >>= 1, o >>= 1) {
    const bool up = (lane & o) != 0;
#pragma unroll
    for (int i = 0; i < half; ++i) {
      const double send = up ? v[i] : v[i + half], keep = up ? v[i + half] : v[i];
      v[i] = keep + __shfl_xor_sync(0xffffffffu, send, o);
    }
  }
  v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
  // best candidate of the warp: the exponent is >= 0 (or +inf), so its bit pattern orders like the value and the
  // minimum is three integer warp reductions (high word, low word, then the lowest index among the ties, A18)
  {
    const unsigned long long kb = (unsigned long long)__double_as_longlong(bv);
    const unsigned hi = (unsigned)(kb >> 32), lo = (unsigned)kb;
    const unsigned mhi = __reduce_min_sync(0xffffffffu, hi);
    const unsigned mlo = __reduce_min_sync(0xffffffffu, hi == mhi ? lo : 0xffffffffu);
    const bool win = hi == mhi && lo == mlo;
    const unsigned mbi = __reduce_min_sync(0xffffffffu, win ? (unsigned)bi : 0xffffffffu);
    const int src = __ffs(__ballot_sync(0xffffffffu, win && (unsigned)bi == mbi)) - 1;
    bn = __shfl_sync(0xffffffffu, bn, src);
    bv = __longlong_as_double((long long)(((unsigned long long)mhi << 32) | mlo));
    bi = (int)mbi;
  }
  if ((lane & 1) == 0 && (lane >> 1) < UP_NQ) sh[warp][lane >> 1] = v[0];
  if (lane == 0) { sh[warp][UP_NQ] = bv; sh[warp][UP_NQ + 1] = (double)bi; sh[warp][UP_NQ + 2] = (double)bn; }
  __syncthreads();
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");     // all CTAs of the cluster have started
  // this CTA's row -> rows[rank] in the first CTA's shared memory
  double* dst = cluster.map_shared_rank(&rows[0][0], 0) + rank * UP_STRIDE;
  if (threadIdx.x < UP_NQ) {
    double s = 0.0;
    for (int w = 0; w < UP_THREADS / 32; ++w) s += sh[w][threadIdx.x];
    dst[threadIdx.x] = s;
  } else if (threadIdx.x == 32) {                          // another warp: runs beside the sums, not after them
    double v = sh[0][UP_NQ], vi = sh[0][UP_NQ + 1], vn = sh[0][UP_NQ + 2];
    for (int w = 1; w < UP_THREADS / 32; ++w)
      if (sh[w][UP_NQ] < v || (sh[w][UP_NQ] == v && sh[w][UP_NQ + 1] < vi)) { v = sh[w][UP_NQ]; vi = sh[w][UP_NQ + 1]; vn = sh[w][UP_NQ + 2]; }
    dst[UP_NQ] = v; dst[UP_NQ + 1] = vi; dst[UP_NQ + 2] = vn;
  }
  cluster.sync();                                         // rows complete and visible in the first CTA
  if (rank != 0) return;
  if (threadIdx.x < UP_NQ) {
    double s = 0.0;
    for (unsigned b = 0; b < C; ++b) s += rows[b][threadIdx.x];
    tot[threadIdx.x] = s;
  } else if (threadIdx.x == 32) {                          // another warp: runs beside the sums, not after them
    double v = rows[0][UP_NQ], vi = rows[0][UP_NQ + 1], vn = rows[0][UP_NQ + 2];
    for (unsigned b = 1; b < C; ++b)
      if (rows[b][UP_NQ] < v || (rows[b][UP_NQ] == v && rows[b][UP_NQ + 1] < vi)) { v = rows[b][UP_NQ]; vi = rows[b][UP_NQ + 1]; vn = rows[b][UP_NQ + 2]; }
    tot[UP_NQ] = v; tot[UP_NQ + 1] = vi; tot[UP_NQ + 2] = vn;
  }
  __syncthreads();
  if (p.row_out) {                                         // sharded evaluation: hand the row to the exchange
    if (threadIdx.x < UP_STRIDE) p.row_out[threadIdx.x] = tot[threadIdx.x];
    if (threadIdx.x == UP_STRIDE) { p.row_out[UP_STRIDE] = rho_ref; p.row_out[UP_STRIDE + 1] = (double)M_O; p.row_out[UP_STRIDE + 2] = 0.0; }
    return;
  }
  if (threadIdx.x != 0) return;
  swarm_serial_step(p, tot, Tin, empty_run_in, r, rho_ref, M_O, total);
}

// Particle-sharded evaluation, second half: every rank folds the rows of all ranks in rank order (same bits on every
// rank) and applies Eq. 15-18, 21 and the stop rules to its own copy of the state.
__global__ void k_swarm_apply(UpdParams p, const double* __restrict__ rows, int G) {
  if (threadIdx.x != 0) return;
  TrackDev* st = p.st;
  if (st->done) return;
  double tot[UP_STRIDE];
  for (int q = 0; q < UP_NQ; ++q) { double s = 0.0; for (int b = 0; b < G; ++b) s += rows[b * UP_ROW + q]; tot[q] = s; }
  double v = rows[UP_NQ], vi = rows[UP_NQ + 1], vn = rows[UP_NQ + 2];
  for (int b = 1; b < G; ++b) {
    const double* rb = rows + b * UP_ROW;
    if (rb[UP_NQ] < v || (rb[UP_NQ] == v && rb[UP_NQ + 1] < vi)) { v = rb[UP_NQ]; vi = rb[UP_NQ + 1]; vn = rb[UP_NQ + 2]; }
  }
  tot[UP_NQ] = v; tot[UP_NQ + 1] = vi; tot[UP_NQ + 2] = vn;
  double Tin[12], r[6];
  for (int a = 0; a < 12; ++a) Tin[a] = st->T[a];
  for (int d = 0; d < 6; ++d) r[d] = st->r[d];
  swarm_serial_step(p, tot, Tin, st->empty_run, r, rows[UP_STRIDE], (int)rows[UP_STRIDE + 1], p.n_total + 1);
}

// End of a frame: state (and trace rows) into the pinned host mirrors.
__global__ void k_track_end(const unsigned long long* __restrict__ st, unsigned long long* __restrict__ st_host, int n_st,
                            const unsigned long long* __restrict__ tr, unsigned long long* __restrict__ tr_host, int n_tr) {
  for (int i = threadIdx.x; i < n_st; i += blockDim.x) st_host[i] = st[i];
  for (int i = threadIdx.x; i < n_tr; i += blockDim.x) tr_host[i] = tr[i];
}

// ---------------------------------------------------------------- host side
struct LoopPlan {
  const rf_pst_set* ps; int M[3]; int iters, k0, has_r0, want_trace, pdl;
  TrackCfg cfg;
};

// k_swarm_update as ONE thread-block cluster of 1, 2, 4 or 8 CTAs (by the number of candidates).
static cudaError_t launch_swarm_update(cudaStream_t st, const UpdParams& up, int N, int pdl) {
  int C = 1;
  while (C < UP_MAX_CLUSTER && C * UP_THREADS < N + 1) C *= 2;
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3(C); cfg.blockDim = dim3(UP_THREADS); cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = C; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = pdl ? 2 : 1;
  return cudaLaunchKernelEx(&cfg, k_swarm_update, up);
}

// Everything of one frame that depends only on library-owned buffers: begin, [A11 init], iters x (fitness, update),
// result copies.  Enqueued on `st`: either the volume's stream directly, or the capture stream when the frame
// loop is being recorded into a CUDA graph.
static int enqueue_loop(rf_volume* v, cudaStream_t st, const LoopPlan& lp) {
  TrackDev* td = v->track;
  const int clear_n = (int)v->acc_cap;
  // the per-call block (poses, r_0) was dropped into init_dev by k_backproject3, as whose kernel arguments it travelled (a copy
  // node here would queue on the host-to-device copy engine behind a caller's prefetch of the next frame, rf_stage_frame, and a
  // read of the pinned host block from the kernel costs a PCIe round trip at the head of the frame)
  k_track_begin<<<(clear_n + 255) / 256, 256, 0, st>>>((const TrackInit*)v->init_dev, td, v->acc[0], v->acc[1], clear_n, v->d_MO);
  RF_LAUNCHED(1);
  MaskCfg mk; mk.mode = (lp.cfg.variant & RF_TRACK_NO_OVERLAP) ? 0 : 1; mk.fx = lp.cfg.fx; mk.fy = lp.cfg.fy; mk.cx = lp.cfg.cx; mk.cy = lp.cfg.cy; mk.w = lp.cfg.w; mk.h = lp.cfg.h;
  int e = 0, rc;
  if (!lp.has_r0) {
    rc = rf_launch_eval(v, st, v->pts_raw[0], lp.M[0], lp.ps->pst_dev[0], 0, 1, td->T, td->r, td->Tprev, mk, nullptr, 0, 0);
    if (rc != RF_OK) return rc;
    k_init_r0<<<1, 32, 0, st>>>(v->acc[0], v->d_MO, td, lp.cfg);
    RF_LAUNCHED(1);
    e = 1;
  }
  for (int k = lp.k0 + 1; k <= lp.k0 + lp.iters; ++k, ++e) {
    const int l = (k - 1) % 3;                           // A15: levels in the listed order, cycling
    const int set = e & 1;
    rc = rf_launch_eval(v, st, v->pts_raw[l], lp.M[l], lp.ps->pst_dev[l], lp.ps->N[l], 1, td->T, td->r, td->Tprev, mk, &td->done, set, lp.pdl);
    if (rc != RF_OK) return rc;
    UpdParams up;
    up.acc = v->acc[set]; up.acc_next = v->acc[set ^ 1]; up.clear_n = clear_n; up.MO = v->d_MO + set; up.MO_next = v->d_MO + (set ^ 1);
    up.N = lp.ps->N[l]; up.pst = lp.ps->pst_dev[l]; up.st = td; up.cfg = lp.cfg; up.k = k; up.k0 = lp.k0; up.level = l;
    up.trace = lp.want_trace ? v->trace_dev : nullptr;
    up.idx_off = 0; up.n_total = lp.ps->N[l]; up.row_out = nullptr;
    rf_prof_begin(v, 3);
    cudaError_t le = launch_swarm_update(st, up, lp.ps->N[l], lp.pdl);
    rf_prof_end(v, 3);
    RF_CUDA(le);
    RF_LAUNCHED(1);
  }
  RF_CUDA(cudaGetLastError());
  // results to the pinned host mirrors by a one-CTA kernel (posted writes over PCIe, complete when the kernel is): a copy node
  // costs the copy engine's start-up on the frame's critical path
  static_assert(sizeof(TrackDev) % 8 == 0 && sizeof(rf_track_trace) % 8 == 0, "copied as 64-bit words");
  k_track_end<<<1, 256, 0, st>>>((const unsigned long long*)td, (unsigned long long*)v->track_host, (int)(sizeof(TrackDev) / 8),
                                 (const unsigned long long*)v->trace_dev, (unsigned long long*)v->trace_host,
                                 lp.want_trace ? (int)(lp.iters * sizeof(rf_track_trace) / 8) : 0);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  return RF_OK;
}

// prelaunch_fusion: enqueue the pose-independent first kernel of this frame's fusion (k_tile_max) behind the frame loop
// and wait for the loop's results on an event, so that kernel runs while the host wakes up (rf_track_integrate).
static int track_impl(rf_volume* v, const rf_frame* f, const rf_pst_set* ps, int32_t iters, rf_track_state* state,
                      rf_track_result* result, rf_track_trace* trace, int prelaunch_fusion) {
  RF_ARG(v && f && ps && state && result, "rf_pfo_track: NULL argument");
  RF_ARG((f->depth || f->depth_on_host == 2) && f->width > 0 && f->height > 0, "rf_pfo_track: bad frame");
  RF_ARG(iters >= 1 && iters <= RF_MAX_ITERS, "rf_pfo_track: iters must be in [1,64]");
  RF_ARG(state->start_iter >= 0 && state->start_iter < 4096, "rf_pfo_track: bad start_iter");
  RF_ARG(state->start_iter == 0 || state->has_r0, "rf_pfo_track: start_iter > 0 needs r0");
  for (int l = 0; l < 3; ++l) {
    RF_ARG(ps->pst_dev[l] && ps->N[l] > 0 && ps->stride[l] > 0, "rf_pfo_track: bad pst_set");
    RF_ARG(ps->stride[l] / 2 < f->width && ps->stride[l] / 2 < f->height, "rf_pfo_track: stride larger than the image");
  }
  cudaStream_t st = v->stream;
  int rc = rf_atlas_sync(v);
  if (rc != RF_OK) return rc;
  const size_t px = (size_t)f->width * f->height;
  const float* d_dev = f->depth;
  if (f->depth_on_host == 2) {
    // the oldest prefetched frame (rf_stage_frame): wait for its copy, then it is the current frame
    RF_ARG(v->pre_count > 0, "rf_pfo_track: no prefetched frame");
    const int slot = v->pre_head;
    RF_ARG(v->pre_w[slot] == f->width && v->pre_h[slot] == f->height, "rf_pfo_track: prefetched frame has another size");
    RF_CUDA(cudaStreamWaitEvent(st, v->pre_done[slot], 0));
    d_dev = v->pre_buf[slot];
    v->pre_head ^= 1; v->pre_count -= 1;
    v->staged_w = f->width; v->staged_h = f->height; v->cur_frame = d_dev;
  } else if (f->depth_on_host) {
    rc = rf_ensure((void**)&v->depth_stage, &v->depth_cap, px * sizeof(float));
    if (rc != RF_OK) return rc;
    RF_CUDA(cudaMemcpyAsync(v->depth_stage, f->depth, px * sizeof(float), cudaMemcpyHostToDevice, st));
    d_dev = v->depth_stage;
    v->staged_w = f->width; v->staged_h = f->height; v->cur_frame = v->depth_stage;
  }
  // a0: the three levels, once per frame (outside the graph: the depth pointer is the caller's)
  rf_prof_begin(v, 5);
  LoopPlan lp;
  lp.ps = ps; lp.iters = iters; lp.k0 = state->start_iter; lp.has_r0 = state->has_r0; lp.want_trace = trace != nullptr;
  lp.pdl = (state->flags & RF_TRACK_NO_PDL) ? 0 : 1;
  for (int l = 0; l < 3; ++l) {
    const int s = ps->stride[l];
    const int nu = (f->width - s / 2 + s - 1) / s, nv = (f->height - s / 2 + s - 1) / s;
    RF_ARG((size_t)nu * nv <= RF_MAX_POINTS, "rf_pfo_track: more than 2^20-1 points in a level");
    const size_t need = (size_t)nu * nv * sizeof(float4);
    if (need > v->pts_cap[l]) {
      cudaFree(v->pts_raw[l]); v->pts_raw[l] = nullptr; v->pts_cap[l] = 0;
      RF_CUDA(cudaMalloc(&v->pts_raw[l], need));
      v->pts_cap[l] = need;
      v->graph_valid = 0;
    }
  }
  TrackInit* in = (TrackInit*)v->init_host;
  for (int a = 0; a < 12; ++a) { in->T[a] = state->pose_c2w[a]; in->Tprev[a] = state->prev_pose_c2w[a]; }
  for (int d = 0; d < 6; ++d) in->r[d] = state->has_r0 ? state->r0[d] : 0.0;
  in->has_r0 = state->has_r0; in->pad = 0;
  in->thresh = ((state->flags & RF_TRACK_THRESH_EQ21) && state->start_iter > 0 && state->aps_threshold > 0.f) ? (double)state->aps_threshold : 0.0;
  rc = rf_launch_backproject3(st, d_dev, f->width, f->height, f->K, ps->stride, v->pts_raw, lp.M, in, v->init_dev);
  if (rc != RF_OK) return rc;
  rf_prof_end(v, 5);
  size_t maxc = 0;
  for (int l = 0; l < 3; ++l) maxc = max(maxc, (size_t)ps->N[l] + 1);
  if (maxc > v->acc_cap) {
    cudaFree(v->acc[0]); cudaFree(v->acc[1]); v->acc[0] = v->acc[1] = nullptr; v->acc_cap = 0;
    RF_CUDA(cudaMalloc(&v->acc[0], (maxc + 1024) * sizeof(unsigned long long)));
    RF_CUDA(cudaMalloc(&v->acc[1], (maxc + 1024) * sizeof(unsigned long long)));
    v->acc_cap = maxc + 1024;
    v->graph_valid = 0;
  }
  lp.cfg.fx = f->K[0]; lp.cfg.fy = f->K[1]; lp.cfg.cx = f->K[2]; lp.cfg.cy = f->K[3]; lp.cfg.w = f->width; lp.cfg.h = f->height;
  RF_ARG(!((state->flags & RF_TRACK_MODE_F1) && (state->flags & RF_TRACK_MODE_EQ14)), "rf_pfo_track: F1 and Eq. 14 are exclusive");
  lp.cfg.mode = (state->flags & RF_TRACK_MODE_F1) ? 1 : (state->flags & RF_TRACK_MODE_EQ14) ? 2 : 0;
  lp.cfg.variant = state->flags & (RF_TRACK_NO_OVERLAP | RF_TRACK_RESCALE_ISO | RF_TRACK_RESCALE_ANISO | RF_TRACK_THRESH_EQ21);
  lp.cfg.early_stop = (state->flags & RF_TRACK_NO_EARLY_STOP) ? 0 : 1;
  lp.cfg.iters = iters;

  const bool use_graph = !v->prof_on && !(state->flags & RF_TRACK_NO_GRAPH);
  if (!use_graph) {
    rc = enqueue_loop(v, st, lp);
    if (rc != RF_OK) return rc;
  } else {
    // signature of everything baked into the captured launches
    unsigned long long sig[16];
    memset(sig, 0, sizeof(sig));
    for (int l = 0; l < 3; ++l) { sig[l] = (unsigned long long)(uintptr_t)ps->pst_dev[l]; sig[3 + l] = ((unsigned long long)ps->N[l] << 32) | (unsigned)lp.M[l]; }
    memcpy(&sig[6], f->K, 16);
    sig[8] = ((unsigned long long)f->width << 32) | (unsigned)f->height;
    sig[9] = ((unsigned long long)iters << 32) | (unsigned)lp.k0;
    sig[10] = ((unsigned long long)lp.has_r0 << 40) | ((unsigned long long)lp.want_trace << 32) | (unsigned)(lp.cfg.variant * 8 + lp.cfg.mode * 2 + lp.cfg.early_stop);
    sig[11] = (unsigned long long)(uintptr_t)v->atlas;
    sig[12] = (unsigned long long)lp.pdl;
    if (!v->graph_valid || memcmp(sig, v->graph_sig, sizeof(sig)) != 0) {
      if (v->graph_exec) { cudaGraphExecDestroy(v->graph_exec); v->graph_exec = nullptr; }
      v->graph_valid = 0;
      RF_CUDA(cudaStreamBeginCapture(v->cap_stream, cudaStreamCaptureModeThreadLocal));
      t_rf_capturing = 1; t_rf_captured = 0;             // captured, not launched: counted apart
      rc = enqueue_loop(v, v->cap_stream, lp);
      t_rf_capturing = 0;
      cudaGraph_t graph = nullptr;
      cudaError_t ce = cudaStreamEndCapture(v->cap_stream, &graph);
      v->graph_launches = (int)t_rf_captured;
      if (rc != RF_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
      if (ce != cudaSuccess) return rf_cuda_fail(ce, "rf_pfo_track: stream capture");
      ce = cudaGraphInstantiate(&v->graph_exec, graph, 0);
      cudaGraphDestroy(graph);
      if (ce != cudaSuccess) return rf_cuda_fail(ce, "rf_pfo_track: graph instantiate");
      memcpy(v->graph_sig, sig, sizeof(sig));
      v->graph_valid = 1;
    }
    RF_CUDA(cudaGraphLaunch(v->graph_exec, st));
    RF_LAUNCHED(v->graph_launches);
  }
  if (prelaunch_fusion && !v->prof_on) {
    if (!v->track_done) RF_CUDA(cudaEventCreateWithFlags(&v->track_done, cudaEventDisableTiming));
    RF_CUDA(cudaEventRecord(v->track_done, st));
    rc = rf_integrate_prelaunch(v, d_dev, f->width, f->height);
    if (rc != RF_OK) return rc;
    RF_CUDA(cudaEventSynchronize(v->track_done));
  } else {
    RF_CUDA(cudaStreamSynchronize(st));
  }
  if (v->prof_on) rf_prof_collect(v);
  const TrackDev& h = *v->track_host;
  for (int a = 0; a < 12; ++a) state->pose_c2w[a] = (float)h.T[a];
  for (int d = 0; d < 6; ++d) state->r0[d] = (float)h.r1[d];
  state->has_r0 = 1;
  state->aps_threshold = (float)h.thresh;
  result->iters_run = h.iters_run; result->status = h.status; result->final_fitness = (float)h.final_rho;
  result->final_count = h.final_count; result->argmax = h.argmax; result->evals = h.evals;
  if (trace) memcpy(trace, v->trace_host, (size_t)h.iters_run * sizeof(rf_track_trace));
  return RF_OK;
}

extern "C" int rf_pfo_track(rf_volume* v, const rf_frame* f, const rf_pst_set* ps, int32_t iters, rf_track_state* state,
                            rf_track_result* result, rf_track_trace* trace) {
  return track_impl(v, f, ps, iters, state, result, trace, 0);
}

// One frame of the paper's pipeline in one call: rf_pfo_track, then rf_integrate_ex of the same frame at the tracked
// pose.  Nothing new is computed; the point is that the fusion kernels are enqueued from C the moment the tracked pose
// is on the host, so the GPU does not idle while a caller's interpreter gets from one call to the next.
extern "C" int rf_track_integrate(rf_volume* v, const rf_frame* f, const rf_pst_set* ps, int32_t iters, rf_track_state* state,
                                  rf_track_result* result, rf_track_trace* trace, const float* gate_center, float gate_radius,
                                  int32_t* integrated_out) {
  RF_ARG(integrated_out, "rf_track_integrate: NULL argument");
  *integrated_out = 0;
  int rc = track_impl(v, f, ps, iters, state, result, trace, 1);
  if (rc != RF_OK) { if (v) v->tile_ready_src = nullptr; return rc; }
  if (gate_center) {
    const float dx = state->pose_c2w[3] - gate_center[0], dy = state->pose_c2w[7] - gate_center[1], dz = state->pose_c2w[11] - gate_center[2];
    if (!(sqrtf(dx * dx + dy * dy + dz * dz) <= gate_radius)) {      // the caller decides what to fuse instead
      v->tile_ready_src = nullptr;
      return RF_OK;
    }
  }
  // the frame's device copy: the caller's pointer, or the staged / prefetched copy rf_pfo_track just consumed
  rc = f->depth_on_host ? rf_integrate_ex(v, nullptr, 2, f->width, f->height, f->K, state->pose_c2w)
                        : rf_integrate_ex(v, f->depth, 0, f->width, f->height, f->K, state->pose_c2w);
  v->tile_ready_src = nullptr;               // never outlives this call
  if (rc != RF_OK) return rc;
  *integrated_out = 1;
  return RF_OK;
}


// ---------------------------------------------------------------- particle-sharded frame loop
// Every rank holds the whole volume and point sets and a slice of each level's template.  Per iteration a rank evaluates
// its slice (+ the centre, which every rank evaluates: same bits everywhere), reduces it to one row of UP_ROW doubles
// (rf_shard_eval); the caller exchanges the rows (one all-gather of 128 bytes per rank: NCCL / gloo, plumbing); every
// rank folds all rows in rank order and applies the update to its own copy of the state (rf_shard_apply).  With one rank
// the result is bit-identical to rf_pfo_track.
struct ShardPlan { int N[3], off[3], Ntot[3], M[3]; const float* pst[3]; TrackCfg cfg; int k0, want_mask; MaskCfg mk; };

extern "C" int rf_shard_begin(rf_volume* v, const rf_frame* f, const rf_pst_set* ps, const int32_t offset[3], const int32_t n_total[3],
                              rf_track_state* state) {
  RF_ARG(v && f && ps && offset && n_total && state, "rf_shard_begin: NULL argument");
  RF_ARG(f->depth && f->depth_on_host == 0 && f->width > 0 && f->height > 0, "rf_shard_begin: the frame must be a device pointer");
  RF_ARG(state->has_r0, "rf_shard_begin: r0 is required (track the first frame with rf_pfo_track)");
  for (int l = 0; l < 3; ++l) {
    RF_ARG(ps->pst_dev[l] && ps->N[l] > 0 && ps->stride[l] > 0 && offset[l] >= 0 && offset[l] + ps->N[l] <= n_total[l], "rf_shard_begin: bad slice");
    RF_ARG(ps->stride[l] / 2 < f->width && ps->stride[l] / 2 < f->height, "rf_shard_begin: stride larger than the image");
  }
  cudaStream_t st = v->stream;
  int rc = rf_atlas_sync(v);
  if (rc != RF_OK) return rc;
  if (!v->shard) { v->shard = calloc(1, sizeof(ShardPlan)); if (!v->shard) { rf_set_error("rf_shard_begin: out of host memory"); return RF_ERR_OOM; } }
  ShardPlan& sp = *(ShardPlan*)v->shard;
  for (int l = 0; l < 3; ++l) {
    const int s = ps->stride[l];
    const int nu = (f->width - s / 2 + s - 1) / s, nv = (f->height - s / 2 + s - 1) / s;
    RF_ARG((size_t)nu * nv <= RF_MAX_POINTS, "rf_shard_begin: more than 2^20-1 points in a level");
    const size_t need = (size_t)nu * nv * sizeof(float4);
    if (need > v->pts_cap[l]) {
      cudaFree(v->pts_raw[l]); v->pts_raw[l] = nullptr; v->pts_cap[l] = 0;
      RF_CUDA(cudaMalloc(&v->pts_raw[l], need));
      v->pts_cap[l] = need; v->graph_valid = 0;
    }
    sp.N[l] = ps->N[l]; sp.off[l] = offset[l]; sp.Ntot[l] = n_total[l]; sp.pst[l] = ps->pst_dev[l];
  }
  rc = rf_launch_backproject3(st, f->depth, f->width, f->height, f->K, ps->stride, v->pts_raw, sp.M, nullptr, nullptr);
  if (rc != RF_OK) return rc;
  size_t maxc = 0;
  for (int l = 0; l < 3; ++l) maxc = max(maxc, (size_t)ps->N[l] + 1);
  if (maxc > v->acc_cap) {
    cudaFree(v->acc[0]); cudaFree(v->acc[1]); v->acc[0] = v->acc[1] = nullptr; v->acc_cap = 0;
    RF_CUDA(cudaMalloc(&v->acc[0], (maxc + 1024) * sizeof(unsigned long long)));
    RF_CUDA(cudaMalloc(&v->acc[1], (maxc + 1024) * sizeof(unsigned long long)));
    v->acc_cap = maxc + 1024; v->graph_valid = 0;
  }
  RF_ARG(!((state->flags & RF_TRACK_MODE_F1) && (state->flags & RF_TRACK_MODE_EQ14)), "rf_shard_begin: F1 and Eq. 14 are exclusive");
  sp.cfg.fx = f->K[0]; sp.cfg.fy = f->K[1]; sp.cfg.cx = f->K[2]; sp.cfg.cy = f->K[3]; sp.cfg.w = f->width; sp.cfg.h = f->height;
  sp.cfg.mode = (state->flags & RF_TRACK_MODE_F1) ? 1 : (state->flags & RF_TRACK_MODE_EQ14) ? 2 : 0;
  sp.cfg.variant = state->flags & (RF_TRACK_NO_OVERLAP | RF_TRACK_RESCALE_ISO | RF_TRACK_RESCALE_ANISO | RF_TRACK_THRESH_EQ21);
  sp.cfg.early_stop = (state->flags & RF_TRACK_NO_EARLY_STOP) ? 0 : 1;
  sp.cfg.iters = RF_MAX_ITERS;
  sp.k0 = 0;
  sp.mk.mode = (sp.cfg.variant & RF_TRACK_NO_OVERLAP) ? 0 : 1; sp.mk.fx = sp.cfg.fx; sp.mk.fy = sp.cfg.fy; sp.mk.cx = sp.cfg.cx; sp.mk.cy = sp.cfg.cy;
  sp.mk.w = sp.cfg.w; sp.mk.h = sp.cfg.h;
  TrackInit* in = (TrackInit*)v->init_host;
  for (int a = 0; a < 12; ++a) { in->T[a] = state->pose_c2w[a]; in->Tprev[a] = state->prev_pose_c2w[a]; }
  for (int d = 0; d < 6; ++d) in->r[d] = state->r0[d];
  in->has_r0 = 1; in->thresh = 0.0;
  const int clear_n = (int)v->acc_cap;
  k_track_begin<<<(clear_n + 255) / 256, 256, 0, st>>>((const TrackInit*)v->init_host, v->track, v->acc[0], v->acc[1], clear_n, v->d_MO);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  return RF_OK;
}

static UpdParams shard_params(rf_volume* v, const ShardPlan& sp, int k) {
  const int l = (k - 1) % 3, set = (k - 1) & 1;
  UpdParams up;
  up.acc = v->acc[set]; up.acc_next = v->acc[set ^ 1]; up.clear_n = (int)v->acc_cap; up.MO = v->d_MO + set; up.MO_next = v->d_MO + (set ^ 1);
  up.N = sp.N[l]; up.pst = sp.pst[l]; up.st = v->track; up.cfg = sp.cfg; up.k = k; up.k0 = 0; up.level = l;
  up.trace = v->trace_dev;                                  // row k - 1: this iteration's trace
  up.idx_off = sp.off[l]; up.n_total = sp.Ntot[l]; up.row_out = nullptr;
  return up;
}

extern "C" int rf_shard_eval(rf_volume* v, int32_t k, double* row_out_dev) {
  RF_ARG(v && v->shard && row_out_dev && k >= 1 && k <= RF_MAX_ITERS, "rf_shard_eval: bad argument (rf_shard_begin first)");
  const ShardPlan& sp = *(const ShardPlan*)v->shard;
  const int l = (k - 1) % 3, set = (k - 1) & 1;
  TrackDev* td = v->track;
  int rc = rf_launch_eval(v, v->stream, v->pts_raw[l], sp.M[l], sp.pst[l], sp.N[l], 1, td->T, td->r, td->Tprev, sp.mk, &td->done, set, 0);
  if (rc != RF_OK) return rc;
  UpdParams up = shard_params(v, sp, k);
  up.row_out = row_out_dev;
  RF_CUDA(launch_swarm_update(v->stream, up, sp.N[l], 0));
  RF_LAUNCHED(1);
  return RF_OK;
}

extern "C" int rf_shard_apply(rf_volume* v, int32_t k, const double* rows_dev, int32_t G, rf_track_trace* trace_row_or_null,
                              int32_t* done_out) {
  RF_ARG(v && v->shard && rows_dev && G >= 1 && k >= 1 && k <= RF_MAX_ITERS && done_out, "rf_shard_apply: bad argument");
  const ShardPlan& sp = *(const ShardPlan*)v->shard;
  UpdParams up = shard_params(v, sp, k);
  k_swarm_apply<<<1, 32, 0, v->stream>>>(up, rows_dev, G);
  RF_CUDA(cudaGetLastError());
  RF_LAUNCHED(1);
  RF_CUDA(cudaMemcpyAsync(v->track_host, v->track, sizeof(TrackDev), cudaMemcpyDeviceToHost, v->stream));
  if (trace_row_or_null) RF_CUDA(cudaMemcpyAsync(v->trace_host, v->trace_dev + (k - 1), sizeof(rf_track_trace), cudaMemcpyDeviceToHost, v->stream));
  RF_CUDA(cudaStreamSynchronize(v->stream));
  if (trace_row_or_null) memcpy(trace_row_or_null, v->trace_host, sizeof(rf_track_trace));
  *done_out = v->track_host->done;
  return RF_OK;
}

extern "C" int rf_shard_end(rf_volume* v, rf_track_state* state, rf_track_result* result) {
  RF_ARG(v && v->shard && state && result, "rf_shard_end: bad argument");
  RF_CUDA(cudaMemcpyAsync(v->track_host, v->track, sizeof(TrackDev), cudaMemcpyDeviceToHost, v->stream));
  RF_CUDA(cudaStreamSynchronize(v->stream));
  const TrackDev& h = *v->track_host;
  for (int a = 0; a < 12; ++a) state->pose_c2w[a] = (float)h.T[a];
  for (int d = 0; d < 6; ++d) state->r0[d] = (float)h.r1[d];
  state->has_r0 = 1;
  state->aps_threshold = (float)h.thresh;
  result->iters_run = h.iters_run; result->status = h.status; result->final_fitness = (float)h.final_rho;
  result->final_count = h.final_count; result->argmax = h.argmax; result->evals = h.evals;
  return RF_OK;
}

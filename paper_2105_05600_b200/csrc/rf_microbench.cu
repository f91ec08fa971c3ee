// rf_microbench.cu -- measurement helper: the L2 roofline denominators.
// MEASURED_PEAKS.json carries no L2 figure, so bench.py measures it in the same run:
//   mode 0  independent uniformly-random 32-byte sector reads over an L2-resident buffer (one 16-byte load
//           per lane at a random sector, 8 independent loads in flight per thread); 32 B counted per request.
//           Both load paths (ld.global.nc through L1TEX, ld.global.cg) are timed and the faster one is reported,
//           so the denominator is the best gather rate this library can demonstrate, not a particular instruction;
//   mode 1  streaming 128-bit reads of the same buffer (same rule).
#include "rf_common.cuh"

template <bool NC> __device__ __forceinline__ uint4 mb_load(const uint4* p) { return NC ? __ldg(p) : __ldcg(p); }

template <bool NC>
__global__ void k_l2_random(const uint4* __restrict__ buf, unsigned nsec, int iters, unsigned* __restrict__ sink) {
  unsigned s = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
  unsigned acc = 0;
  for (int it = 0; it < iters; ++it) {
    uint4 v[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      s = s * 1664525u + 1013904223u;                      // LCG: address stream independent of the data
      const unsigned sec = __umulhi(s, nsec);               // uniform over [0, nsec) for any sector count
      v[q] = mb_load<NC>(buf + (size_t)sec * 2);           // 32-byte sector = two uint4; read the first
    }
#pragma unroll
    for (int q = 0; q < 8; ++q) acc ^= v[q].x ^ v[q].w;
  }
  if (acc == 0x9e3779b9u) sink[0] = acc;
}

template <bool NC>
__global__ void k_l2_stream(const uint4* __restrict__ buf, size_t n16, int iters, unsigned* __restrict__ sink) {
  unsigned acc = 0;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (int it = 0; it < iters; ++it)
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) {
      const uint4 v = mb_load<NC>(buf + i);
      acc ^= v.x ^ v.w;
    }
  if (acc == 0x9e3779b9u) sink[0] = acc;
}

extern "C" int rf_microbench_l2(int64_t bytes, int32_t mode, int32_t reps, double* gbps_out) {
  RF_ARG(gbps_out && bytes >= (1 << 20) && reps > 0, "rf_microbench_l2: bad argument");
  RF_ARG(bytes / 32 < 0xffffffffll, "rf_microbench_l2: at most 2^32 sectors");
  const size_t nsec = (size_t)(bytes / 32);                // exactly the requested size, in 32-byte sectors
  const size_t nbytes = nsec * 32;
  uint4* buf = nullptr; unsigned* sink = nullptr;
  RF_CUDA(cudaMalloc(&buf, nbytes));
  RF_CUDA(cudaMalloc(&sink, 4));
  RF_CUDA(cudaMemset(buf, 1, nbytes));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int blocks = 148 * 8, threads = 256, iters = 64;
  double best = 0;
  for (int r = 0; r < 2 * (reps + 2); ++r) {
    const bool nc = (r & 1) != 0;
    cudaEventRecord(e0);
    if (mode == 0) { if (nc) k_l2_random<true><<<blocks, threads>>>(buf, (unsigned)nsec, iters, sink); else k_l2_random<false><<<blocks, threads>>>(buf, (unsigned)nsec, iters, sink); }
    else { if (nc) k_l2_stream<true><<<blocks, threads>>>(buf, nbytes / 16, 8, sink); else k_l2_stream<false><<<blocks, threads>>>(buf, nbytes / 16, 8, sink); }
    cudaEventRecord(e1);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) { cudaFree(buf); cudaFree(sink); return rf_cuda_fail(e, "rf_microbench_l2"); }
    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
    const double moved = mode == 0 ? (double)blocks * threads * iters * 8 * 32.0 : (double)nbytes * 8;
    if (r >= 4) best = fmax(best, moved / (ms * 1e-3) / 1e9);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(buf); cudaFree(sink);
  *gbps_out = best;
  return RF_OK;
}

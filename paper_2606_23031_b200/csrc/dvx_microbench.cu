// dvx_microbench.cu - the machine's fp32 FMA / instruction-issue rate, measured in the same run as the benchmark
// ("measured FMA peak from a micro-benchmark in the same run").  The compositing kernels of the hot
// path are bound by instruction issue, not by HBM; this is the denominator of that roofline.
// One FFMA per lane per clock per SM sub-partition is both the fp32 peak and the issue peak (one warp instruction per
// clock per sub-partition), so one kernel measures both.
#include "dvx_internal.cuh"

namespace {

constexpr int MB_THREADS = 256, MB_CHAINS = 16, MB_UNROLL = 4;

// 16 independent FFMA chains per thread (enough to cover the 4-cycle dependent-issue latency at any occupancy), the loop
// body unrolled 4 x: 64 FFMA per 3 loop instructions.  The result is stored so that nothing is optimised away.
__global__ void __launch_bounds__(MB_THREADS) fma_issue_kernel(float *out, uint32_t iters, float a, float b) {
  float x[MB_CHAINS];
#pragma unroll
  for (int i = 0; i < MB_CHAINS; ++i) x[i] = (float)(threadIdx.x + i) * 1e-3f;
  for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < MB_UNROLL; ++u)
#pragma unroll
      for (int i = 0; i < MB_CHAINS; ++i) x[i] = fmaf(x[i], a, b);
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < MB_CHAINS; ++i) s += x[i];
  out[(size_t)blockIdx.x * MB_THREADS + threadIdx.x] = s;
}

}  // namespace

// Launches the kernel on `blocks` CTAs; returns the FFMA count per thread (= iters * 64).
uint64_t dvx_microbench_fma_launch(float *out, uint32_t blocks, uint32_t iters, cudaStream_t st) {
  DVX_COUNT_LAUNCH(1);
  fma_issue_kernel<<<blocks, MB_THREADS, 0, st>>>(out, iters, 0.999f, 1e-3f);
  return (uint64_t)iters * MB_CHAINS * MB_UNROLL;
}
uint32_t dvx_microbench_threads(void) { return MB_THREADS; }

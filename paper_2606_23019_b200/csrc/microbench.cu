// microbench.cu -- sa_debug_ex2_rate: the measured MUFU.EX2 rate of this GPU, the roofline
// denominator of sa_block_significance (K4: 16 384 exponentials per 128 x 128 tile against
// 512 clk of MMA, so the special-function pipe bounds that kernel). A measurement hook for bench.py,
// not part of the method: every resident warp runs eight independent ex2.approx chains, nothing else
// competes for the pipe, so the rate is what the hardware can sustain at the clock it holds under
// that load.
#include "common.cuh"

namespace sa {
namespace {

constexpr int kThreads = 256;
constexpr int kChains = 8;

__global__ void __launch_bounds__(kThreads) ex2_rate_kernel(float* __restrict__ sink, int iters) {
  float y[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) y[i] = 0.001f * (threadIdx.x + 1) + 0.1f * i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < kChains; ++i) {
      float r;
      asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(-y[i]));   // y in (0, 1] -> [0.5, 1)
      y[i] = r;
    }
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += y[i];
  if (s == 12345.678f) sink[blockIdx.x] = s;     // never true: keeps the chains alive
}

}  // namespace

cudaError_t launch_ex2_rate(int iters, float* sink, int n_sm, cudaStream_t st, double* n_exp) {
  const int grid = n_sm * 8;                     // 2048 threads per SM: every warp slot taken
  ex2_rate_kernel<<<grid, kThreads, 0, st>>>(sink, iters);
  *n_exp = static_cast<double>(grid) * kThreads * kChains * static_cast<double>(iters);
  return cudaGetLastError();
}

}  // namespace sa

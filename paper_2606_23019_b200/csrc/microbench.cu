// microbench.cu -- sa_debug_ex2_rate: the measured MUFU.EX2 rate of this GPU, the roofline
// denominator of sa_block_significance (K4: 16 384 exponentials per 128 x 128 tile against
// 512 clk of MMA, so the special-function pipe bounds that kernel). A measurement hook for bench.py,
// not part of the method: every resident warp runs eight independent ex2.approx chains, nothing else
// competes for the pipe, so the rate is what the hardware can sustain at the clock it holds under
// that load.
#include "common.cuh"
#include "ptx.cuh"

namespace sa {
namespace {
using namespace ptx;

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

// L2 -> shared-memory fill rate, the secondary bound of the attention kernel on masks whose work items
// share no key blocks (K1: an unshared (tile, key block) unit needs a 32 KB K tile and a
// 32 KB V tile of its own). One CTA per SM; one warp keeps kFillSlots bulk copies of 32 KB in flight
// into a shared-memory ring (cp.async.bulk, completion on an mbarrier per slot: the mechanism the
// attention kernel's TMA loads use, without a tensor map), nothing consumes the data. The CTAs walk
// the buffer tile by tile, all of them together, so a buffer that fits L2 is served from L2 after the
// first pass, like the K and V of the one or two heads the attention kernel has in flight.
constexpr int kFillSlots = 6;
constexpr uint32_t kFillTile = 32768;
__global__ void __launch_bounds__(32, 1)
l2_fill_kernel(const unsigned char* __restrict__ buf, unsigned n_tiles, int iters) {
  extern __shared__ __align__(1024) unsigned char fill_smem[];
  __shared__ uint64_t full[kFillSlots];
  const int lane = threadIdx.x;
  if (lane == 0) {
    for (int s = 0; s < kFillSlots; ++s) mbar_init(smem_u32(&full[s]), 1);
    fence_mbar_init();
  }
  __syncwarp();
  const uint32_t base = smem_u32(fill_smem);
  unsigned tile = blockIdx.x % n_tiles;
  for (int i = 0; i < iters + kFillSlots; ++i) {
    const int s = i % kFillSlots;
    if (i >= kFillSlots) mbar_wait(smem_u32(&full[s]), ((i / kFillSlots) - 1) & 1);   // the slot's previous copy
    if (i < iters) {
      mbar_expect_tx_e(smem_u32(&full[s]), kFillTile);
      const unsigned char* src = buf + static_cast<size_t>(tile) * kFillTile;
      asm volatile(
          "{\n\t.reg .pred e;\n\telect.sync _|e, 0xffffffff;\n\t"
          "@e cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n\t}"
          ::"r"(base + s * kFillTile), "l"(src), "r"(kFillTile), "r"(smem_u32(&full[s]))
          : "memory");
      tile += gridDim.x;
      if (tile >= n_tiles) tile -= n_tiles * (tile / n_tiles);
    }
  }
}

}  // namespace

cudaError_t launch_l2_fill(const void* buf, size_t buf_bytes, int iters, int n_sm, cudaStream_t st,
                           double* bytes_moved) {
  const unsigned n_tiles = static_cast<unsigned>(buf_bytes / kFillTile);
  if (n_tiles == 0) return cudaErrorInvalidValue;
  const int smem = kFillSlots * kFillTile + 1024;
  cudaError_t e = ensure_dynamic_smem(kSmemL2Fill, reinterpret_cast<const void*>(l2_fill_kernel), smem);
  if (e != cudaSuccess) return e;
  l2_fill_kernel<<<n_sm, 32, smem, st>>>(static_cast<const unsigned char*>(buf), n_tiles, iters);
  *bytes_moved = static_cast<double>(n_sm) * iters * kFillTile;
  return cudaGetLastError();
}

cudaError_t launch_ex2_rate(int iters, float* sink, int n_sm, cudaStream_t st, double* n_exp) {
  const int grid = n_sm * 8;                     // 2048 threads per SM: every warp slot taken
  ex2_rate_kernel<<<grid, kThreads, 0, st>>>(sink, iters);
  *n_exp = static_cast<double>(grid) * kThreads * kChains * static_cast<double>(iters);
  return cudaGetLastError();
}

}  // namespace sa

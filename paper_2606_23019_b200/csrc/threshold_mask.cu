// threshold_mask.cu -- sa_mask_from_threshold: the paper's own run-time mask path.
//
// M_p = 1(T <= p) (Sec. 4.1.2; Alg. 1 l.31) of a per-head threshold map
// kept at a BASE resolution, instantiated at the TARGET resolution by the conservative bilinear
// resize with a ceiling rule (Sec. 4.3.1, Eq. 7):
//     R_target(u,v) = ceil( Phi(R_base, u / s_h, v / s_w) ),   R_base = 1(T_base <= p*_h),
// and written straight into CRM bit-rows (LSB-first).
//
// ceil of a bilinear blend of 0/1 values is 1 exactly when a base cell with POSITIVE weight is
// active (readings P14-P16), so no floating-point interpolation is needed: with
// x = u * nbq / NQB the cell a0 = floor(x) always has positive weight and a0 + 1 has one iff
// (u * nbq) % NQB != 0 (clamped at the last cell); likewise along v. All of it is integer work, so
// the result is bit-exact by construction. One warp produces one 32-bit mask word per step with
// __ballot_sync; lanes read consecutive key blocks (coalesced). HBM/L2-bound streaming: the map
// is read once (up to 4 neighbouring cells per target block, which share cache lines).
#include "common.cuh"

namespace sa {
namespace {

constexpr int kThreads = 256;

// one warp per bit-row (h, u): the two base rows are fixed for the row; 32-bit index arithmetic
// (the host side bounds the sizes so that u * nbq and v * nbk stay below 2^31). Measured at the
// 480p -> 720p shape (H = 40): 49 us per call; one warp per mask WORD was slower (90 us: the
// per-word index divisions dominate), so the row form stays.
__global__ void __launch_bounds__(kThreads)
mask_from_threshold_kernel(const float* __restrict__ tmap, const float* __restrict__ p_star,
                           uint32_t* __restrict__ mask_bits, int H, int nbq, int nbk, int NQB,
                           int NKB, int W, int force_diag) {
  const int lane = threadIdx.x & 31;
  const int n_rows = H * NQB;            // < 2^31 (checked by the caller)
  const int warp0 = (blockIdx.x * kThreads + threadIdx.x) >> 5;
  const int n_warps = (gridDim.x * kThreads) >> 5;
  for (int r = warp0; r < n_rows; r += n_warps) {
    const int h = r / NQB, u = r - h * NQB;
    const float p = __ldg(p_star + h);
    const uint32_t xu = static_cast<uint32_t>(u) * static_cast<uint32_t>(nbq);
    const int a0 = static_cast<int>(xu / static_cast<uint32_t>(NQB));
    const bool two_rows = (xu % static_cast<uint32_t>(NQB) != 0u) && (a0 + 1 < nbq);
    const float* row0 = tmap + (static_cast<size_t>(h) * nbq + a0) * nbk;
    const float* row1 = two_rows ? row0 + nbk : row0;
    uint32_t* dst = mask_bits + static_cast<size_t>(r) * W;
#pragma unroll 4
    for (int wv = 0; wv < W; ++wv) {
      const int v = wv * 32 + lane;
      bool on = false;
      if (v < NKB) {
        const uint32_t yv = static_cast<uint32_t>(v) * static_cast<uint32_t>(nbk);
        const int b0 = static_cast<int>(yv / static_cast<uint32_t>(NKB));
        const bool two_cols = (yv % static_cast<uint32_t>(NKB) != 0u) && (b0 + 1 < nbk);
        on = __ldg(row0 + b0) <= p;
        if (two_cols) on = on || __ldg(row0 + b0 + 1) <= p;
        if (two_rows) {
          on = on || __ldg(row1 + b0) <= p;
          if (two_cols) on = on || __ldg(row1 + b0 + 1) <= p;
        }
        if (force_diag && u == v) on = true;
      }
      const uint32_t bits = __ballot_sync(0xFFFFFFFFu, on);
      if (lane == 0) dst[wv] = bits;
    }
  }
}

}  // namespace

cudaError_t launch_mask_from_threshold(const float* tmap, const float* p_star, uint32_t* mask_bits,
                                       int H, int nbq, int nbk, int NQB, int NKB, int force_diag,
                                       cudaStream_t st) {
  const int W = (NKB + 31) / 32;
  const long long n_rows = static_cast<long long>(H) * NQB;
  long long blocks = (n_rows * 32 + kThreads - 1) / kThreads;
  const long long cap = 148LL * 8 * 4;     // grid-stride beyond 4 waves of 8 resident CTAs per SM
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  mask_from_threshold_kernel<<<static_cast<unsigned>(blocks), kThreads, 0, st>>>(
      tmap, p_star, mask_bits, H, nbq, nbk, NQB, NKB, W, force_diag);
  return cudaGetLastError();
}

}  // namespace sa

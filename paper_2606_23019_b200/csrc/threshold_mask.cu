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
// the result is bit-exact by construction.
//
// Layout of the work (HBM/L2-bound streaming; the map is 10.5 MB and the mask 1.8 MB at H = 40,
// 256 x 256 -> 591 x 591): a CTA takes 32 target rows of one head. The column map v -> (b0, second
// column?) does not depend on the row: it is computed once per CTA into shared memory (one integer
// division per target column per CTA instead of two per mask bit). A warp then takes a target row:
// it reads the row's one or two base rows with coalesced loads, compares with p* and ORs them into
// a packed bit-row in shared memory (__ballot_sync), and every target bit is two shared-memory
// lookups into that bit-row. Mask words are written 32 at a time (one coalesced store per 32 words).
#include "common.cuh"

namespace sa {
namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kRowsPerBlock = 32;

// dynamic shared memory: uint16 colmap[NKB] (b0 | second column << 15), then per warp nbw =
// ceil(nbk / 32) words of the ORed base bit-row
__global__ void __launch_bounds__(kThreads)
mask_from_threshold_kernel(const float* __restrict__ tmap, const float* __restrict__ p_star,
                           uint32_t* __restrict__ mask_bits, int nbq, int nbk, int NQB, int NKB, int W,
                           int force_diag) {
  extern __shared__ uint32_t s_dyn[];
  const int nbw = (nbk + 31) / 32;
  uint32_t* s_bits = s_dyn;                                          // [kWarps][nbw]
  uint16_t* s_col = reinterpret_cast<uint16_t*>(s_dyn + kWarps * nbw);   // [NKB]
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int h = blockIdx.y;
  for (int v = threadIdx.x; v < NKB; v += kThreads) {
    const uint32_t yv = static_cast<uint32_t>(v) * static_cast<uint32_t>(nbk);   // < 2^31 (host check)
    const uint32_t b0 = yv / static_cast<uint32_t>(NKB);
    const bool two = (yv - b0 * static_cast<uint32_t>(NKB) != 0u) && (b0 + 1u < static_cast<uint32_t>(nbk));
    s_col[v] = static_cast<uint16_t>(b0 | (two ? 0x8000u : 0u));
  }
  __syncthreads();
  const float p = __ldg(p_star + h);
  uint32_t* my_bits = s_bits + warp * nbw;
  const int u_end = min((blockIdx.x + 1) * kRowsPerBlock, NQB);
  for (int u = blockIdx.x * kRowsPerBlock + warp; u < u_end; u += kWarps) {
    const uint32_t xu = static_cast<uint32_t>(u) * static_cast<uint32_t>(nbq);
    const uint32_t a0 = xu / static_cast<uint32_t>(NQB);
    const bool two_rows = (xu - a0 * static_cast<uint32_t>(NQB) != 0u) && (a0 + 1u < static_cast<uint32_t>(nbq));
    const float* row0 = tmap + (static_cast<size_t>(h) * nbq + a0) * nbk;
    const float* row1 = two_rows ? row0 + nbk : row0;
    // active base cells of the row's one or two base rows, ORed, as packed bits
    // (16 loads in flight per lane: the pass is latency-bound otherwise)
    for (int wb0 = 0; wb0 < nbw; wb0 += 8) {
      float x0[8], x1[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int b = (wb0 + i) * 32 + lane;
        const bool in = b < nbk;
        x0[i] = in ? __ldg(row0 + b) : INFINITY;
        x1[i] = in ? __ldg(row1 + b) : INFINITY;
      }
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const uint32_t x = __ballot_sync(0xFFFFFFFFu, x0[i] <= p || x1[i] <= p);
        if (lane == 0 && wb0 + i < nbw) my_bits[wb0 + i] = x;
      }
    }
    __syncwarp();
    uint32_t* dst = mask_bits + (static_cast<size_t>(h) * NQB + u) * W;
    for (int w0 = 0; w0 < W; w0 += 32) {
      uint32_t mine = 0u;
      const int wn = min(32, W - w0);
      for (int i = 0; i < wn; ++i) {
        const int v = (w0 + i) * 32 + lane;
        bool on = false;
        if (v < NKB) {
          const uint32_t c = s_col[v];
          const uint32_t b0 = c & 0x7FFFu;
          on = (my_bits[b0 >> 5] >> (b0 & 31u)) & 1u;
          if (c & 0x8000u) on = on || ((my_bits[(b0 + 1u) >> 5] >> ((b0 + 1u) & 31u)) & 1u);
          if (force_diag && u == v) on = true;
        }
        const uint32_t x = __ballot_sync(0xFFFFFFFFu, on);
        if (lane == i) mine = x;
      }
      if (lane < wn) dst[w0 + lane] = mine;
    }
    __syncwarp();                                  // my_bits is rewritten for the warp's next row
  }
}

}  // namespace

cudaError_t launch_mask_from_threshold(const float* tmap, const float* p_star, uint32_t* mask_bits,
                                       int H, int nbq, int nbk, int NQB, int NKB, int force_diag,
                                       cudaStream_t st) {
  const int W = (NKB + 31) / 32;
  const size_t smem = static_cast<size_t>(kWarps) * ((nbk + 31) / 32) * 4 + static_cast<size_t>(NKB) * 2;
  if (smem > 48 * 1024) {
    cudaError_t e = ensure_dynamic_smem(kSmemMaskFromThreshold,
                                        reinterpret_cast<const void*>(mask_from_threshold_kernel), 100 * 1024);
    if (e != cudaSuccess) return e;
  }
  const dim3 grid((NQB + kRowsPerBlock - 1) / kRowsPerBlock, H);
  mask_from_threshold_kernel<<<grid, kThreads, smem, st>>>(tmap, p_star, mask_bits, nbq, nbk, NQB, NKB, W,
                                                          force_diag);
  return cudaGetLastError();
}

}  // namespace sa

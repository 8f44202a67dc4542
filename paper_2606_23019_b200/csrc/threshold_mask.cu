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
// Layout of the work (the map is 10.5 MB and the mask 1.8 MB at H = 40, 256 x 256 -> 591 x 591): a CTA
// takes 16 target rows of one head. Everything about a target column that does not depend on the row
// (word and bit of its one or two base columns) is computed once per CTA into shared memory, one word
// per column (one integer division per column per CTA instead of two per mask bit). The base rows the
// CTA's target rows touch are compared with p* and packed into bit-rows in shared memory ONCE per CTA
// (coalesced reads, eight loads in flight per lane, __ballot_sync). A warp then takes a target row:
// the OR of its one or two base bit-rows sits in a register per lane (up to 1024 base columns; in
// shared memory beyond), and a target bit is two shuffles away. Mask words are written 32 at a time.
// The kernel is bound by its own instruction count (~12 instructions per mask bit-word lane), not by
// bandwidth: 24 us at that shape (round 1: one warp per row with four dependent gathers and two
// divisions per bit, 49 us).
#include "common.cuh"

namespace sa {
namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kRowsPerBlock = 16;

// dynamic shared memory: s_rows[n_rows_cap][nbw] packed base bit-rows (1(T <= p*) of the base rows this
// CTA's target rows touch, each compared and packed ONCE per CTA), then uint16 colmap[NKB]
// (b0 | second column << 15). If the CTA's base-row span does not fit n_rows_cap (a strong downscale),
// the rows are packed per target row into the first kWarps bit-rows instead.
__global__ void __launch_bounds__(kThreads)
mask_from_threshold_kernel(const float* __restrict__ tmap, const float* __restrict__ p_star,
                           uint32_t* __restrict__ mask_bits, int nbq, int nbk, int NQB, int NKB, int W,
                           int force_diag, int n_rows_cap) {
  extern __shared__ uint32_t s_dyn[];
  const int nbw = (nbk + 31) / 32;
  uint32_t* s_rows = s_dyn;                                              // [n_rows_cap][nbw]
  uint32_t* s_col = s_dyn + n_rows_cap * nbw;                            // [NKB]
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int h = blockIdx.y;
  const float p = __ldg(p_star + h);
  const int u_first = blockIdx.x * kRowsPerBlock;
  const int u_end = min(u_first + kRowsPerBlock, NQB);
  // base rows the CTA's target rows touch: a0(u_first) .. a0(u_end - 1) + 1
  const uint32_t a_lo = static_cast<uint32_t>(u_first) * static_cast<uint32_t>(nbq) / static_cast<uint32_t>(NQB);
  const uint32_t a_hi = min(static_cast<uint32_t>(u_end - 1) * static_cast<uint32_t>(nbq) / static_cast<uint32_t>(NQB) + 1u,
                            static_cast<uint32_t>(nbq - 1));
  const int n_rows = static_cast<int>(a_hi - a_lo) + 1;
  const bool shared_rows = n_rows <= n_rows_cap;

  // pack (a) 8 words of one base row per call: 8 loads in flight per lane, then 8 ballots
  auto pack8 = [&](const float* row, int wb0, uint32_t* dst, bool or_into) {
    float x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int b = (wb0 + i) * 32 + lane;
      x[i] = b < nbk ? __ldg(row + b) : INFINITY;
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const uint32_t bits = __ballot_sync(0xFFFFFFFFu, x[i] <= p);
      if (lane == 0 && wb0 + i < nbw) dst[wb0 + i] = or_into ? (dst[wb0 + i] | bits) : bits;
    }
  };
  if (shared_rows) {
    // (row, 8-word group) pairs dealt to the warps: every base row is read and compared once per CTA
    const int groups = (nbw + 7) / 8;
    for (int job = warp; job < n_rows * groups; job += kWarps) {
      const int r = job / groups, g8 = job - r * groups;
      pack8(tmap + (static_cast<size_t>(h) * nbq + a_lo + r) * nbk, g8 * 8, s_rows + r * nbw, false);
    }
  }
  for (int v = threadIdx.x; v < NKB; v += kThreads) {
    const uint32_t yv = static_cast<uint32_t>(v) * static_cast<uint32_t>(nbk);   // < 2^31 (host check)
    const uint32_t b0 = yv / static_cast<uint32_t>(NKB);
    const bool two = (yv - b0 * static_cast<uint32_t>(NKB) != 0u) && (b0 + 1u < static_cast<uint32_t>(nbk));
    // everything about column v that does not depend on the row, in one word: word and bit of its
    // first base column [0,15), the same for the second one [15,30), "has a second column" (bit 31)
    const uint32_t b1 = two ? b0 + 1u : b0;
    s_col[v] = (b0 >> 5) | ((b0 & 31u) << 10) | ((b1 >> 5) << 15) | ((b1 & 31u) << 25);
  }
  __syncthreads();
  for (int u = u_first + warp; u < u_end; u += kWarps) {
    const uint32_t xu = static_cast<uint32_t>(u) * static_cast<uint32_t>(nbq);
    const uint32_t a0 = xu / static_cast<uint32_t>(NQB);
    const bool two_rows = (xu - a0 * static_cast<uint32_t>(NQB) != 0u) && (a0 + 1u < static_cast<uint32_t>(nbq));
    const uint32_t *r0, *r1;              // packed bits of the row's one or two base rows
    if (shared_rows) {
      r0 = s_rows + (a0 - a_lo) * nbw;
      r1 = two_rows ? r0 + nbw : r0;
    } else {
      uint32_t* mine = s_rows + warp * nbw;       // n_rows_cap >= kWarps
      const float* row0 = tmap + (static_cast<size_t>(h) * nbq + a0) * nbk;
      for (int wb0 = 0; wb0 < nbw; wb0 += 8) {
        pack8(row0, wb0, mine, false);
        if (two_rows) {
          __syncwarp();
          pack8(row0 + nbk, wb0, mine, true);
        }
      }
      __syncwarp();
      r0 = r1 = mine;
    }
    uint32_t* dst = mask_bits + (static_cast<size_t>(h) * NQB + u) * W;
    // the OR of the row's base bit-rows: in a register per lane when it has at most 32 words (a target
    // bit is then two shuffles away), else looked up in shared memory
    const bool in_regs = nbw <= 32;
    const uint32_t rc = (in_regs && lane < nbw) ? (r0[lane] | r1[lane]) : 0u;
    for (int w0 = 0; w0 < W; w0 += 32) {
      uint32_t mine_w = 0u;
      const int wn = min(32, W - w0);
      for (int i = 0; i < wn; ++i) {
        const int v = (w0 + i) * 32 + lane;
        const uint32_t c = v < NKB ? s_col[v] : 0u;
        const uint32_t i0 = c & 1023u, s0 = (c >> 10) & 31u, i1 = (c >> 15) & 1023u, s1 = c >> 25;
        uint32_t x0, x1;
        if (in_regs) {
          x0 = __shfl_sync(0xFFFFFFFFu, rc, static_cast<int>(i0));
          x1 = __shfl_sync(0xFFFFFFFFu, rc, static_cast<int>(i1));
        } else {
          x0 = r0[i0] | r1[i0];
          x1 = r0[i1] | r1[i1];
        }
        bool on = (((x0 >> s0) | (x1 >> s1)) & 1u) != 0u;
        if (force_diag && u == v) on = true;
        const uint32_t x = __ballot_sync(0xFFFFFFFFu, on && v < NKB);
        if (lane == i) mine_w = x;
      }
      if (lane < wn) dst[w0 + lane] = mine_w;
    }
    __syncwarp();                                  // (per-row mode) the warp's bit-row is rewritten next
  }
}

}  // namespace

cudaError_t launch_mask_from_threshold(const float* tmap, const float* p_star, uint32_t* mask_bits,
                                       int H, int nbq, int nbk, int NQB, int NKB, int force_diag,
                                       cudaStream_t st) {
  const int W = (NKB + 31) / 32;
  // shared memory: as many packed base rows as a CTA's 32 target rows can touch (32 * nbq / NQB + 2), if
  // that fits beside the column map; else the per-warp rows only
  const size_t nbw = (nbk + 31) / 32;
  const size_t col_bytes = static_cast<size_t>(NKB) * 4;
  long long n_rows_cap = (static_cast<long long>(kRowsPerBlock) * nbq + NQB - 1) / NQB + 2;
  if (n_rows_cap < kWarps) n_rows_cap = kWarps;
  if (static_cast<size_t>(n_rows_cap) * nbw * 4 + col_bytes > 160 * 1024) n_rows_cap = kWarps;
  const size_t smem = static_cast<size_t>(n_rows_cap) * nbw * 4 + col_bytes;
  if (smem > 48 * 1024) {
    cudaError_t e = ensure_dynamic_smem(kSmemMaskFromThreshold,
                                        reinterpret_cast<const void*>(mask_from_threshold_kernel), 164 * 1024);
    if (e != cudaSuccess) return e;
  }
  const dim3 grid((NQB + kRowsPerBlock - 1) / kRowsPerBlock, H);
  mask_from_threshold_kernel<<<grid, kThreads, smem, st>>>(tmap, p_star, mask_bits, nbq, nbk, NQB, NKB, W,
                                                          force_diag, static_cast<int>(n_rows_cap));
  return cudaGetLastError();
}

}  // namespace sa

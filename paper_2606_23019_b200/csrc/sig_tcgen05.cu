// sig_tcgen05.cu -- sa_block_significance: WEST's block-wise aggregation (Sec. 4.1.1,
// Eq. 1; Alg. 1 l.9-10) without materialising the attention matrix:
//     S(u,v) = (1/B^2) * sum_{p in B_u} sum_{q in B_v} A(p,q),   A(p,q) = exp(scale*q_p.k_q - lse_p)
// where lse is what a density-1 call of the forward pass has already written. Per (head, query
// block) the kernel is the QK^T half of the forward pass: every key block's S = Q K^T goes to TMEM
// (tcgen05.mma, operands staged by TMA, 128B swizzle), a softmax warpgroup reads it, evaluates
// exp2(s*c - lse2) (log2 domain, one FFMA + one MUFU per element), sums the 128 x 128 tile and
// writes ONE float. There is no P, no PV and no running max (lse is final), so the two S buffers
// ping-pong freely: the MMA of tile v+1 runs under the exponentials of tile v. The exponentials
// (16 384 per tile at 16/clk/SM = 1024 clk) bound it, not the 512 clk MMA.
//
// Persistent grid, one CTA per SM; work items (b, h, query block) in head-major order with a static
// stride (all items cost the same). Warp 0: TMA producer, warp 1: MMA issuer (both converged, elect.sync
// issue), warp 2: TMEM allocator, warps 4-7 / 8-11: warpgroup 0 / 1, which take the even / odd
// tiles. Padded keys (>= n_valid) get zero weight, padded query rows are left out (P18).
#include <cuda.h>

#include "common.cuh"
#include "ptx.cuh"

namespace sa {
namespace {

using namespace ptx;

constexpr int kBlk = 128;
constexpr int kD = 128;
constexpr int kThreads = 384;
constexpr uint32_t kTileBytes = kBlk * kD * 2;      // 32 KB
constexpr uint32_t kHalfBytes = kTileBytes / 2;
constexpr int kSlots = 6;                           // K ring
constexpr uint32_t kTmemCols = 256;                 // two fp32 128 x 128 S buffers
#ifndef SA_SIG_POLY_PAIRS
#define SA_SIG_POLY_PAIRS 1
#endif
constexpr int kSigPolyPairs = SA_SIG_POLY_PAIRS;    // of every 4 column pairs, how many take exp2 on the FMA pipe
                                                    // (measured at C3: 0 -> 12.94 ms, 1 -> 12.32 ms, 2 -> 14.36 ms)

constexpr uint32_t kOffQ = 0;
constexpr uint32_t kOffRing = kTileBytes;
constexpr uint32_t kOffCtl = kOffRing + kSlots * kTileBytes;
struct __align__(8) Ctl {
  uint64_t q_full, q_empty;
  uint64_t k_full[kSlots], k_empty[kSlots];
  uint64_t s_full[2], s_free[2];
  float partial[2][2][4];     // [warpgroup][tile parity][warp]: row-sum partials of one tile
  uint32_t tmem_base;
};
constexpr uint32_t kSmemBytes = kOffCtl + sizeof(Ctl);
static_assert(kSmemBytes <= 232448, "exceeds 227 KB of dynamic shared memory");

// K-major 128B-swizzled operand descriptor and bf16 x bf16 -> fp32 128 x 128 instruction descriptor
// (same encodings as fwd_tcgen05.cu)
constexpr uint64_t kDescKMajor = (uint64_t(1) << 16) | (uint64_t(1024 >> 4) << 32) |
                                 (uint64_t(1) << 46) | (uint64_t(2) << 61);
__device__ __forceinline__ uint64_t make_desc(uint32_t smem_addr) {
  return kDescKMajor | static_cast<uint64_t>((smem_addr & 0x3FFFFu) >> 4);
}
constexpr uint32_t kIdescQK = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 3) << 17) |
                              ((128u >> 4) << 24);

struct SigParams {
  const float* lse;
  float* sig;
  int N, n_valid, NQB, NKB, n_items;     // n_items = B * H * NQB
  float scale_log2;
};

struct Ring {
  int slot = 0;
  uint32_t phase = 0;
  __device__ __forceinline__ void advance() {
    if (++slot == kSlots) { slot = 0; phase ^= 1u; }
  }
};

// ------------------------------------------------------------------ warp 0: TMA producer
__device__ void producer(const SigParams& p, Ctl* ctl, uint32_t smem_base, const CUtensorMap* tm_q,
                         const CUtensorMap* tm_k) {
  Ring ring;
  uint32_t q_phase = 0;
  for (int item = blockIdx.x; item < p.n_items; item += gridDim.x) {
    const int bh = item / p.NQB, u = item - bh * p.NQB;
    const int row0 = bh * p.N;
    mbar_wait(smem_u32(&ctl->q_empty), q_phase ^ 1u, 1);
    const uint32_t qf = smem_u32(&ctl->q_full);
    mbar_expect_tx_e(qf, kTileBytes);
    tma_load_2d_e(smem_base + kOffQ, tm_q, 0, row0 + u * kBlk, qf);
    tma_load_2d_e(smem_base + kOffQ + kHalfBytes, tm_q, 64, row0 + u * kBlk, qf);
    q_phase ^= 1u;
    for (int v = 0; v < p.NKB; ++v) {
      const uint32_t full = smem_u32(&ctl->k_full[ring.slot]);
      mbar_wait(smem_u32(&ctl->k_empty[ring.slot]), ring.phase ^ 1u, 2);
      mbar_expect_tx_e(full, kTileBytes);
      const uint32_t dst = smem_base + kOffRing + ring.slot * kTileBytes;
      tma_load_2d_e(dst, tm_k, 0, row0 + v * kBlk, full);
      tma_load_2d_e(dst + kHalfBytes, tm_k, 64, row0 + v * kBlk, full);
      ring.advance();
    }
  }
  mbar_wait(smem_u32(&ctl->q_empty), q_phase ^ 1u, 3);   // every MMA reading smem has retired
}

// ------------------------------------------------------------------ warp 1: MMA issuer
__device__ void mma_issuer(const SigParams& p, Ctl* ctl, uint32_t smem_base, uint32_t tmem) {
  Ring ring;
  uint32_t q_phase = 0, w = 0;           // w: tile counter over all items; tile w uses S buffer w & 1
  for (int item = blockIdx.x; item < p.n_items; item += gridDim.x) {
    mbar_wait(smem_u32(&ctl->q_full), q_phase, 10);
    q_phase ^= 1u;
    for (int v = 0; v < p.NKB; ++v, ++w) {
      const uint32_t buf = w & 1u;
      mbar_wait(smem_u32(&ctl->s_free[buf]), ((w >> 1) & 1u) ^ 1u, 11);   // softmax has read tile w-2
      mbar_wait(smem_u32(&ctl->k_full[ring.slot]), ring.phase, 12);
      tc_fence_after();
      const uint32_t q_addr = smem_base + kOffQ;
      const uint32_t k_addr = smem_base + kOffRing + ring.slot * kTileBytes;
#pragma unroll
      for (int kk = 0; kk < kD / 16; ++kk) {
        const uint32_t off = (kk >> 2) * kHalfBytes + (kk & 3) * 32;
        mma_ss_e(tmem + buf * 128, make_desc(q_addr + off), make_desc(k_addr + off), kIdescQK, kk > 0);
      }
      tc_commit_e(smem_u32(&ctl->s_full[buf]));
      tc_commit_e(smem_u32(&ctl->k_empty[ring.slot]));
      ring.advance();
    }
    tc_commit_e(smem_u32(&ctl->q_empty));
  }
}

// ------------------------------------------------------------------ warps 4-11: exponentials + tile sums
// Warpgroup g takes the tiles with (w & 1) == g; one thread per query row.
__device__ void sum_wg(const SigParams& p, Ctl* ctl, uint32_t tmem, int g, int quarter, int lane) {
  const int row = quarter * 32 + lane;
  const uint32_t tm_s = tmem + (static_cast<uint32_t>(quarter * 32) << 16) + g * 128;
  const float c = p.scale_log2;
  const uint64_t c2 = pk2(c, c);
  uint32_t w = 0;
  for (int item = blockIdx.x; item < p.n_items; item += gridDim.x) {
    const int bh = item / p.NQB, u = item - bh * p.NQB;
    const int qrow = u * kBlk + row;
    // lse in the log2 domain; padded query rows (and rows without any key) contribute nothing
    const float lse = __ldg(p.lse + static_cast<size_t>(bh) * p.N + qrow);
    const bool row_on = qrow < p.n_valid && lse > -INFINITY;
    const float nl2 = row_on ? -lse * 1.4426950408889634f : 0.f;
    const uint64_t nl22 = pk2(nl2, nl2);
    float* out = p.sig + (static_cast<size_t>(bh) * p.NQB + u) * p.NKB;
    for (int v = 0; v < p.NKB; ++v, ++w) {
      if ((w & 1u) != static_cast<uint32_t>(g)) continue;
      const uint32_t par = (w >> 1) & 1u;
      mbar_wait(smem_u32(&ctl->s_full[g]), par, 20);
      tc_fence_after();
      uint32_t sr[4][32];
#pragma unroll
      for (int cc = 0; cc < 4; ++cc) tmem_ld32(tm_s + cc * 32, sr[cc]);
      tc_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctl->s_free[g]));      // S is in registers: buffer free
      const int kv = p.n_valid - v * kBlk;                        // valid keys in this tile
      uint64_t acc[4] = {0ull, 0ull, 0ull, 0ull};
      if (kv >= kBlk) {
#pragma unroll
        for (int cc = 0; cc < 4; ++cc)
#pragma unroll
          for (int i = 0; i < 16; ++i) {
            const uint64_t x = fma2(pk2(__uint_as_float(sr[cc][2 * i]), __uint_as_float(sr[cc][2 * i + 1])),
                                    c2, nl22);
            float e0, e1;
            if ((i & 3) < kSigPolyPairs) {             // FMA-pipe exp2: this kernel is MUFU-bound
              exp2_fma_pipe(x, e0, e1);
            } else {
              float x0, x1;
              up2(x, x0, x1);
              e0 = ex2(x0);
              e1 = ex2(x1);
            }
            acc[i & 3] = add2(acc[i & 3], pk2(e0, e1));
          }
      } else {                                                    // the ragged tail tile
#pragma unroll
        for (int cc = 0; cc < 4; ++cc)
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            const float e = ex2(fmaf(__uint_as_float(sr[cc][i]), c, nl2));
            acc[i & 3] = add2(acc[i & 3], pk2(cc * 32 + i < kv ? e : 0.f, 0.f));
          }
      }
      float a0, a1, b0, b1;
      up2(add2(acc[0], acc[1]), a0, a1);
      up2(add2(acc[2], acc[3]), b0, b1);
      float rs = row_on ? (a0 + a1) + (b0 + b1) : 0.f;
#pragma unroll
      for (int s = 16; s > 0; s >>= 1) rs += __shfl_xor_sync(0xFFFFFFFFu, rs, s);
      if (lane == 0) ctl->partial[g][par][quarter] = rs;
      asm volatile("bar.sync %0, 128;" ::"r"(1 + g) : "memory");   // the 4 warps of this warpgroup
      if (quarter == 0 && lane == 0) {
        const float* pt = ctl->partial[g][par];
        out[v] = ((pt[0] + pt[1]) + (pt[2] + pt[3])) * (1.f / (kBlk * kBlk));
      }
    }
  }
}

__global__ void __launch_bounds__(kThreads, 1)
sig_tcgen05_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                   const SigParams p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t smem_base = smem_u32(smem_raw);
  if (smem_base & 1023u) __trap();   // 128B-swizzled TMA / UMMA tiles need a 1024 B aligned base
  Ctl* ctl = reinterpret_cast<Ctl*>(smem_raw + kOffCtl);
  // warp index through a shuffle: the compiler then knows it is warp-uniform, and the role code below runs on the
  // uniform datapath (see fwd_tcgen05.cu)
  const int warp = __shfl_sync(0xFFFFFFFFu, static_cast<int>(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    prefetch_tensormap(&tm_q);
    prefetch_tensormap(&tm_k);
    mbar_init(smem_u32(&ctl->q_full), 1);
    mbar_init(smem_u32(&ctl->q_empty), 1);
    for (int s = 0; s < kSlots; ++s) {
      mbar_init(smem_u32(&ctl->k_full[s]), 1);
      mbar_init(smem_u32(&ctl->k_empty[s]), 1);
    }
    for (int b = 0; b < 2; ++b) {
      mbar_init(smem_u32(&ctl->s_full[b]), 1);
      mbar_init(smem_u32(&ctl->s_free[b]), 4);    // one arrival per warp of the warpgroup
    }
    fence_mbar_init();
  }
  if (warp == 2) {
    tmem_alloc(smem_u32(&ctl->tmem_base), kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = ctl->tmem_base;
  if (warp < 4) {
    setmaxnreg_dec<88>();
    if (warp == 0) producer(p, ctl, smem_base, &tm_q, &tm_k);
    else if (warp == 1) mma_issuer(p, ctl, smem_base, tmem);
  } else {
    setmaxnreg_inc<208>();
    sum_wg(p, ctl, tmem, warp >= 8 ? 1 : 0, warp & 3, lane);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem, kTmemCols);
}

}  // namespace

cudaError_t launch_block_significance(const __nv_bfloat16* q, const __nv_bfloat16* k, const float* lse,
                                      float* sig, int B, int H, int N, int n_valid, float scale,
                                      cudaStream_t st, const char** err_text) {
  int n_sm = 0;
  cudaError_t e = device_sm_count(&n_sm);
  if (e != cudaSuccess) return e;
  e = ensure_dynamic_smem(kSmemSigTcgen05, reinterpret_cast<const void*>(sig_tcgen05_kernel),
                          static_cast<int>(kSmemBytes));
  if (e != cudaSuccess) { *err_text = "cudaFuncSetAttribute(sig_tcgen05_kernel)"; return e; }
  CUtensorMap tq, tk;
  const uint64_t rows = static_cast<uint64_t>(B) * H * N;
  if (!make_tile_map_128x64(&tq, q, rows) || !make_tile_map_128x64(&tk, k, rows)) {
    *err_text = "cuTensorMapEncodeTiled failed";
    return cudaErrorInvalidValue;
  }
  SigParams p;
  p.lse = lse;
  p.sig = sig;
  p.N = N;
  p.n_valid = n_valid;
  p.NQB = N / kBlk;
  p.NKB = N / kBlk;
  p.n_items = B * H * p.NQB;
  p.scale_log2 = scale * 1.4426950408889634f;
  const int grid = p.n_items < n_sm ? p.n_items : n_sm;
  sig_tcgen05_kernel<<<grid, kThreads, kSmemBytes, st>>>(tq, tk, p);
  return cudaGetLastError();
}

}  // namespace sa

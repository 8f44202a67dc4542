// fwd_mma_sync.cu -- block-sparse attention forward, warp-level mma.sync variant.
//
// The crm kernel (Sec. 4.3.2): FlashAttention forward with the dense KV-block
// iterator replaced by the CRM bit-row iterator (Alg. 2). One CTA owns one
// (batch, head, query block); it walks its bit-row and, for every ACTIVE key block only, stages
// K and V in shared memory (cp.async, double buffered), computes S = Q K^T with bf16 tensor-core
// MMAs (fp32 accumulate), applies the online-softmax update, and accumulates O += P V.
//
// This is the variant that serves (D,Bq,Bk) = (64,64,64) (the tiny correctness shape, for which
// a 64-row tcgen05 tile is not worth a second TMEM layout) and, via sa_set_fwd_variant(1), a
// second CUDA implementation of the (128,128,128) shape for cross-checking the tcgen05 kernel.
// It is a CUDA kernel on the product path, not a CPU fallback.
//
// Layout: each warp owns 16 query rows; mma.sync.m16n8k16 (bf16 in, fp32 accumulate). Shared
// tiles are [rows][D] bf16 with the 16-byte chunk index XOR-swizzled by (row & 7) so that
// ldmatrix reads are bank-conflict free.
#include "common.cuh"

namespace sa {
namespace {

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst), "l"(src));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}
__device__ __forceinline__ void ldmatrix_x4(uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3,
                                            uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];\n"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t& r0, uint32_t& r1, uint32_t& r2,
                                                  uint32_t& r3, uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];\n"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0,
                                               uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, "
      "{%8,%9}, {%0,%1,%2,%3};\n"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 t = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&t);
}

// byte offset of 16-byte chunk `c` of row `r` in a [rows][D] bf16 tile, XOR-swizzled
template <int D>
__device__ __forceinline__ uint32_t tile_off(int r, int c) {
  return static_cast<uint32_t>(r * (D * 2) + ((c ^ (r & 7)) << 4));
}

template <int ROWS, int D, int THREADS>
__device__ __forceinline__ void load_tile_async(uint32_t smem_base, const __nv_bfloat16* gsrc) {
  constexpr int CHUNKS_PER_ROW = D / 8;
  constexpr int TOTAL = ROWS * CHUNKS_PER_ROW;
  static_assert(TOTAL % THREADS == 0, "tile must divide evenly");
#pragma unroll
  for (int i = 0; i < TOTAL / THREADS; ++i) {
    const int idx = threadIdx.x + i * THREADS;
    const int r = idx / CHUNKS_PER_ROW, c = idx % CHUNKS_PER_ROW;
    cp_async16(smem_base + tile_off<D>(r, c), gsrc + static_cast<size_t>(r) * D + c * 8);
  }
}

template <int BLK, int D>
__global__ void __launch_bounds__(BLK * 2, 1) fwd_mma_sync_kernel(const FwdParams p) {
  constexpr int THREADS = BLK * 2;        // one warp per 16 query rows
  constexpr int NT_S = BLK / 8;           // n-tiles of S per warp (keys)
  constexpr int NT_O = D / 8;             // n-tiles of O per warp (head dim)
  constexpr int KS_QK = D / 16;           // k-steps of Q K^T
  constexpr int KS_PV = BLK / 16;         // k-steps of P V
  constexpr uint32_t TILE_BYTES = BLK * D * 2;

  extern __shared__ __align__(128) uint8_t smem[];
  const uint32_t sQ = smem_u32(smem);
  const uint32_t sK0 = sQ + TILE_BYTES;            // K[2]
  const uint32_t sV0 = sK0 + 2 * TILE_BYTES;       // V[2]

  const int4 item = p.items[blockIdx.x];       // single-row items: x = b*H + h, y = query block | 0xFFFF << 16
  const int bh = item.x, u = item.y & 0xFFFF;
  const int h = bh % p.H;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane >> 2, t = lane & 3;

  const size_t head_off = static_cast<size_t>(bh) * p.N * D;
  const __nv_bfloat16* gQ = p.q + head_off + static_cast<size_t>(u) * BLK * D;
  const __nv_bfloat16* gK = p.k + head_off;
  const __nv_bfloat16* gV = p.v + head_off;

  CrmIter it;
  it.init(p.mask_bits + (static_cast<size_t>(h) * p.NQB + u) * p.W, p.W, p.NKB);

  // prologue: Q and the first active K/V block
  load_tile_async<BLK, D, THREADS>(sQ, gQ);
  int v_cur = it.index();
  if (v_cur >= 0) {
    load_tile_async<BLK, D, THREADS>(sK0, gK + static_cast<size_t>(v_cur) * BLK * D);
    load_tile_async<BLK, D, THREADS>(sV0, gV + static_cast<size_t>(v_cur) * BLK * D);
  }
  cp_async_commit();

  float o_acc[NT_O][4];
#pragma unroll
  for (int i = 0; i < NT_O; ++i) o_acc[i][0] = o_acc[i][1] = o_acc[i][2] = o_acc[i][3] = 0.f;
  float m_run[2] = {-INFINITY, -INFINITY};   // running max (log2 domain) of rows g and g+8
  float l_run[2] = {0.f, 0.f};               // running sum (this thread's columns only)

  const int row0 = warp * 16;
  int buf = 0;
  while (v_cur >= 0) {
    it.next();
    const int v_next = it.index();
    if (v_next >= 0) {
      const uint32_t nb = (buf ^ 1) * TILE_BYTES;
      load_tile_async<BLK, D, THREADS>(sK0 + nb, gK + static_cast<size_t>(v_next) * BLK * D);
      load_tile_async<BLK, D, THREADS>(sV0 + nb, gV + static_cast<size_t>(v_next) * BLK * D);
    }
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();

    const uint32_t sK = sK0 + buf * TILE_BYTES, sV = sV0 + buf * TILE_BYTES;

    // ---- S = Q K^T (16 x BLK per warp) ----
    float s_acc[NT_S][4];
#pragma unroll
    for (int i = 0; i < NT_S; ++i) s_acc[i][0] = s_acc[i][1] = s_acc[i][2] = s_acc[i][3] = 0.f;
#pragma unroll
    for (int ks = 0; ks < KS_QK; ++ks) {
      uint32_t a[4];
      {
        const int r = row0 + (lane & 7) + ((lane >> 3) & 1) * 8;
        const int c = ks * 2 + (lane >> 4);
        ldmatrix_x4(a[0], a[1], a[2], a[3], sQ + tile_off<D>(r, c));
      }
#pragma unroll
      for (int np = 0; np < NT_S / 2; ++np) {
        uint32_t b0, b1, b2, b3;
        const int mi = lane >> 3;
        const int r = np * 16 + (lane & 7) + (mi >> 1) * 8;
        const int c = ks * 2 + (mi & 1);
        ldmatrix_x4(b0, b1, b2, b3, sK + tile_off<D>(r, c));
        mma_bf16_16816(s_acc[2 * np], a, b0, b1);
        mma_bf16_16816(s_acc[2 * np + 1], a, b2, b3);
      }
    }

    // ---- padding: keys >= n_valid carry zero weight (only the last key block can hold any) ----
    const int key0 = v_cur * BLK;
    if (key0 + BLK > p.n_valid) {
#pragma unroll
      for (int nt = 0; nt < NT_S; ++nt) {
        const int col = key0 + nt * 8 + 2 * t;
        if (col >= p.n_valid) { s_acc[nt][0] = -INFINITY; s_acc[nt][2] = -INFINITY; }
        if (col + 1 >= p.n_valid) { s_acc[nt][1] = -INFINITY; s_acc[nt][3] = -INFINITY; }
      }
    }

    // ---- online softmax (log2 domain: p = 2^(s*scale*log2e - m)) ----
    float mx[2] = {-INFINITY, -INFINITY};
#pragma unroll
    for (int nt = 0; nt < NT_S; ++nt) {
      mx[0] = fmaxf(mx[0], fmaxf(s_acc[nt][0], s_acc[nt][1]));
      mx[1] = fmaxf(mx[1], fmaxf(s_acc[nt][2], s_acc[nt][3]));
    }
    float alpha[2], m_use[2];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      mx[r] = fmaxf(mx[r], __shfl_xor_sync(0xFFFFFFFFu, mx[r], 1));
      mx[r] = fmaxf(mx[r], __shfl_xor_sync(0xFFFFFFFFu, mx[r], 2));
      const float m_new = fmaxf(m_run[r], mx[r] * p.scale_log2);
      m_use[r] = (m_new == -INFINITY) ? 0.f : m_new;
      alpha[r] = exp2f(m_run[r] - m_use[r]);     // m_run = -inf -> 0
      m_run[r] = m_new;
      l_run[r] *= alpha[r];
    }
#pragma unroll
    for (int nt = 0; nt < NT_O; ++nt) {
      o_acc[nt][0] *= alpha[0]; o_acc[nt][1] *= alpha[0];
      o_acc[nt][2] *= alpha[1]; o_acc[nt][3] *= alpha[1];
    }
#pragma unroll
    for (int nt = 0; nt < NT_S; ++nt) {
      s_acc[nt][0] = exp2f(fmaf(s_acc[nt][0], p.scale_log2, -m_use[0]));
      s_acc[nt][1] = exp2f(fmaf(s_acc[nt][1], p.scale_log2, -m_use[0]));
      s_acc[nt][2] = exp2f(fmaf(s_acc[nt][2], p.scale_log2, -m_use[1]));
      s_acc[nt][3] = exp2f(fmaf(s_acc[nt][3], p.scale_log2, -m_use[1]));
      l_run[0] += s_acc[nt][0] + s_acc[nt][1];
      l_run[1] += s_acc[nt][2] + s_acc[nt][3];
    }

    // ---- O += P V ----
#pragma unroll
    for (int ks = 0; ks < KS_PV; ++ks) {
      uint32_t a[4];
      a[0] = pack_bf16(s_acc[2 * ks][0], s_acc[2 * ks][1]);
      a[1] = pack_bf16(s_acc[2 * ks][2], s_acc[2 * ks][3]);
      a[2] = pack_bf16(s_acc[2 * ks + 1][0], s_acc[2 * ks + 1][1]);
      a[3] = pack_bf16(s_acc[2 * ks + 1][2], s_acc[2 * ks + 1][3]);
#pragma unroll
      for (int np = 0; np < NT_O / 2; ++np) {
        uint32_t b0, b1, b2, b3;
        const int mi = lane >> 3;
        const int r = ks * 16 + (lane & 7) + (mi & 1) * 8;
        const int c = np * 2 + (mi >> 1);
        ldmatrix_x4_trans(b0, b1, b2, b3, sV + tile_off<D>(r, c));
        mma_bf16_16816(o_acc[2 * np], a, b0, b1);
        mma_bf16_16816(o_acc[2 * np + 1], a, b2, b3);
      }
    }
    __syncthreads();   // everyone is done with buf before it is refilled
    buf ^= 1;
    v_cur = v_next;
  }
  cp_async_wait<0>();

  // ---- epilogue: O / l -> bf16, lse = ln2 * (m + log2 l); empty row -> 0 / -inf ----
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    l_run[r] += __shfl_xor_sync(0xFFFFFFFFu, l_run[r], 1);
    l_run[r] += __shfl_xor_sync(0xFFFFFFFFu, l_run[r], 2);
  }
  const float inv0 = l_run[0] > 0.f ? 1.f / l_run[0] : 0.f;
  const float inv1 = l_run[1] > 0.f ? 1.f / l_run[1] : 0.f;
  const int qrow0 = u * BLK + row0 + g;
  __nv_bfloat16* o0 = p.out + head_off + static_cast<size_t>(qrow0) * D;
  __nv_bfloat16* o1 = o0 + 8 * D;
#pragma unroll
  for (int nt = 0; nt < NT_O; ++nt) {
    const int col = nt * 8 + 2 * t;
    *reinterpret_cast<uint32_t*>(o0 + col) = pack_bf16(o_acc[nt][0] * inv0, o_acc[nt][1] * inv0);
    *reinterpret_cast<uint32_t*>(o1 + col) = pack_bf16(o_acc[nt][2] * inv1, o_acc[nt][3] * inv1);
  }
  if (t == 0) {
    float* lse = p.lse + static_cast<size_t>(bh) * p.N + qrow0;
    lse[0] = l_run[0] > 0.f ? 0.6931471805599453f * (m_run[0] + log2f(l_run[0])) : -INFINITY;
    lse[8] = l_run[1] > 0.f ? 0.6931471805599453f * (m_run[1] + log2f(l_run[1])) : -INFINITY;
  }
}

template <int BLK, int D>
cudaError_t launch(const FwdParams& p, cudaStream_t st) {
  constexpr size_t smem = 5ull * BLK * D * 2;
  cudaError_t e = ensure_dynamic_smem(BLK == 64 ? kSmemFwdMmaSync64 : kSmemFwdMmaSync128,
                                      reinterpret_cast<const void*>(fwd_mma_sync_kernel<BLK, D>),
                                      static_cast<int>(smem));
  if (e != cudaSuccess) return e;
  fwd_mma_sync_kernel<BLK, D><<<p.n_items, BLK * 2, smem, st>>>(p);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_fwd_mma_sync(const FwdParams& p, cudaStream_t st, int* n_launch) {
  *n_launch += 1;
  if (p.Bq == 64 && p.D == 64) return launch<64, 64>(p, st);
  if (p.Bq == 128 && p.D == 128) return launch<128, 128>(p, st);
  return cudaErrorInvalidValue;
}

}  // namespace sa

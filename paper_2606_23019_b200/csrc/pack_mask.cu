// pack_mask.cu -- sa_pack_mask: per-head top-fraction selection of block scores -> CRM bits.
//
// Mask instantiation M_p = 1(T <= p) (Sec. 4.1.2; Alg. 1 l.31) in the
// form BASELINE.json names: head h keeps the k_h best-scoring blocks of its NQB x NKB grid
// (readings P1-P4), written as CRM bit-rows (bit order PAPER.md:512,536).
//
// Exact selection without sorting: scores map to order-preserving uint32 keys; an 8-bit-per-pass
// radix select finds the k_h-th largest key T of the head (4 histogram passes over the scores,
// which are L2-resident: 56 MB at the 720p shape); keys > T are kept, and of the keys == T the
// first r in flat-index order, r = k_h - #(keys > T). Index order needs a prefix count of the
// ties: one per-row tie count pass, then each row's warp sums the rows before it and walks its
// own row 32 key blocks at a time with __ballot_sync, which is also what packs the bits. When all
// keys equal to T are kept (T unique: the usual case) both the tie counts and the prefix are skipped.
// Bandwidth/ALU work only; no tensor cores (HBM/L2-bound streaming, coalesced 128 B per warp).
#include "common.cuh"

namespace sa {
namespace {

constexpr int kHistThreads = 256;
constexpr int kHistRowsPerBlock = 16;     // rows of one head per histogram block (2 per warp)

struct HeadState {      // per head, per pass p = 0..3: state after resolving passes < p
  uint32_t prefix[5];   // high bits fixed so far (prefix[p] has the top 8*p bits set)
  uint32_t k_rem[5];    // how many keys with that prefix (ranked from the largest) still to take
  uint32_t n_equal;     // after the last pass: how many keys equal T = prefix[4] the head holds
};

// workspace: hist uint32 [H][4][256] | HeadState [H] | row_ties uint32 [H][NQB]
struct PackWs {
  uint32_t* hist;
  HeadState* state;
  uint32_t* row_ties;
};
__host__ __device__ inline size_t align256(size_t x) { return (x + 255) / 256 * 256; }

PackWs carve(void* ws, int H, int NQB) {
  char* p = static_cast<char*>(ws);
  PackWs w;
  w.hist = reinterpret_cast<uint32_t*>(p);
  p += align256(static_cast<size_t>(H) * 4 * 256 * sizeof(uint32_t));
  w.state = reinterpret_cast<HeadState*>(p);
  p += align256(static_cast<size_t>(H) * sizeof(HeadState));
  w.row_ties = reinterpret_cast<uint32_t*>(p);
  (void)NQB;
  return w;
}

// fp32 score -> uint32 key, larger score <=> larger key. -0 is canonicalised to +0 (x + 0.0f);
// NaN sorts lowest (key 0); a forced diagonal entry takes the top key.
__device__ __forceinline__ uint32_t score_key(float x, bool forced) {
  if (forced) return 0xFFFFFFFFu;
  if (x != x) return 0u;
  x = x + 0.0f;
  const uint32_t b = __float_as_uint(x);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

// k_h = clamp(floor((double)density * total + 0.5), 1, total), raised to the diagonal count when
// forced (P2, P3). Separate fp64 multiply and add, exactly as the definition reads.
__device__ __forceinline__ uint32_t keep_count(float density, int NQB, int NKB, int force_diag) {
  const double total = static_cast<double>(NQB) * static_cast<double>(NKB);
  double kd = floor(__dadd_rn(__dmul_rn(static_cast<double>(density), total), 0.5));
  if (!(kd >= 1.0)) kd = 1.0;
  if (kd > total) kd = total;
  uint32_t k = static_cast<uint32_t>(kd);
  if (force_diag) k = max(k, static_cast<uint32_t>(min(NQB, NKB)));
  return k;
}

// Resolve pass `pass - 1` from its histogram: find the byte value whose bin holds the k_rem-th
// largest key, extend the prefix, reduce k_rem. Called by every block (cheap, 256 bins); the
// result lands in shared memory, and block 0 of the head records it for later kernels.
__device__ void resolve(int pass, int h, const float* density, int NQB, int NKB, int force_diag,
                        const uint32_t* hist, HeadState* state, uint32_t* s_prefix,
                        uint32_t* s_krem, bool record, uint32_t* s_nequal = nullptr) {
  __shared__ uint32_t s_suffix[256];
  if (pass == 0) {
    if (threadIdx.x == 0) {
      *s_prefix = 0u;
      *s_krem = keep_count(density[h], NQB, NKB, force_diag);
      if (record) { state[h].prefix[0] = 0u; state[h].k_rem[0] = *s_krem; }
    }
    __syncthreads();
    return;
  }
  const uint32_t* hh = hist + (static_cast<size_t>(h) * 4 + (pass - 1)) * 256;
  const uint32_t prev_prefix = state[h].prefix[pass - 1];
  const uint32_t prev_krem = state[h].k_rem[pass - 1];
  if (threadIdx.x < 256) s_suffix[threadIdx.x] = hh[threadIdx.x];
  __syncthreads();
  if (threadIdx.x < 32) {
    // bins from the largest byte down until the cumulative count reaches k_rem: lane l owns the 8
    // bins 255-8l .. 248-8l; a warp scan gives the count above each lane's group
    const int lane = threadIdx.x;
    uint32_t c[8], sum = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      c[i] = s_suffix[255 - 8 * lane - i];
      sum += c[i];
    }
    uint32_t incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, incl, o);
      if (lane >= o) incl += t;
    }
    uint32_t above = incl - sum;                       // keys in bins above this lane's group
    const bool here = above < prev_krem && incl >= prev_krem;
    const uint32_t who = __ballot_sync(0xFFFFFFFFu, here);
    // nobody reaches k_rem (cannot happen for a consistent histogram): fall to bin 0 like the walk
    const int owner = who ? __ffs(who) - 1 : 31;
    if (lane == owner) {
      int bin = 255 - 8 * lane;
      int i = 0;
      for (; i < 7; ++i, --bin) {
        if (above + c[i] >= prev_krem) break;
        above += c[i];
      }
      if (!who) {                                      // walk semantics: stop at bin 0 whatever it holds
        bin = 0;
        above = incl - c[7];
      }
      const int shift = 32 - 8 * pass;
      *s_prefix = prev_prefix | (static_cast<uint32_t>(bin) << shift);
      *s_krem = prev_krem - above;
      if (record) {
        state[h].prefix[pass] = *s_prefix;
        state[h].k_rem[pass] = *s_krem;
        if (pass == 4) state[h].n_equal = s_suffix[bin];   // the bin of the full key
      }
      if (s_nequal) *s_nequal = s_suffix[bin];
    }
  }
  __syncthreads();
}

// Histogram of byte `pass` (from the top) of the keys whose higher bytes equal the prefix.
template <int PASS>
__global__ void __launch_bounds__(kHistThreads)
pack_hist_kernel(const float* __restrict__ scores, const float* __restrict__ density, int NQB,
                 int NKB, int force_diag, uint32_t* __restrict__ hist, HeadState* state) {
  __shared__ uint32_t s_hist[256];
  __shared__ uint32_t s_prefix, s_krem;
  const int h = blockIdx.y;
  resolve(PASS, h, density, NQB, NKB, force_diag, hist, state, &s_prefix, &s_krem,
          blockIdx.x == 0);
  for (int i = threadIdx.x; i < 256; i += blockDim.x) s_hist[i] = 0u;
  __syncthreads();
  const uint32_t prefix = s_prefix;
  constexpr int shift = 24 - 8 * PASS;
  const uint32_t hi_mask = PASS == 0 ? 0u : (0xFFFFFFFFu << (32 - 8 * PASS));
  // one warp per row (no index division: the row and column are loop variables), lanes on
  // consecutive columns (coalesced)
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int row0 = blockIdx.x * kHistRowsPerBlock;
  const int row1 = min(row0 + kHistRowsPerBlock, NQB);
  for (int u = row0 + warp; u < row1; u += kHistThreads / 32) {
    const float* row = scores + (static_cast<size_t>(h) * NQB + u) * NKB;
    for (int v0 = 0; v0 < NKB; v0 += 128) {       // four loads in flight per lane (L2 latency)
      float x[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int v = v0 + q * 32 + lane;
        x[q] = v < NKB ? __ldg(row + v) : 0.f;
      }
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int v = v0 + q * 32 + lane;
        bool hit = false;
        uint32_t bin = 0u;
        if (v < NKB) {
          const uint32_t key = score_key(x[q], force_diag && u == v);
          hit = (key & hi_mask) == prefix;
          bin = (key >> shift) & 0xFFu;
        }
        if (PASS == 0) {           // top byte: a handful of values -> merge equal bins in the warp
          const uint32_t active = __ballot_sync(0xFFFFFFFFu, hit);
          if (hit) {
            const uint32_t same = __match_any_sync(active, bin);
            if (lane == __ffs(same) - 1) atomicAdd(&s_hist[bin], static_cast<uint32_t>(__popc(same)));
          }
        } else if (hit) {          // lower bytes: bins are spread (match.any would loop per value)
          atomicAdd(&s_hist[bin], 1u);
        }
      }
    }
  }
  __syncthreads();
  uint32_t* hh = hist + (static_cast<size_t>(h) * 4 + PASS) * 256;
  for (int i = threadIdx.x; i < 256; i += blockDim.x)
    if (s_hist[i]) atomicAdd(hh + i, s_hist[i]);
}

// After pass 3: T = full key of the k_h-th largest, r = ties to keep. One warp per row counts the
// keys equal to T in its row. grid = (ceil(NQB/8), H), 8 warps per block.
__global__ void __launch_bounds__(256)
pack_row_ties_kernel(const float* __restrict__ scores, const float* __restrict__ density, int NQB,
                     int NKB, int force_diag, const uint32_t* __restrict__ hist, HeadState* state,
                     uint32_t* __restrict__ row_ties) {
  __shared__ uint32_t s_T, s_r, s_neq;
  const int h = blockIdx.y;
  resolve(4, h, density, NQB, NKB, force_diag, hist, state, &s_T, &s_r, blockIdx.x == 0, &s_neq);
  const uint32_t T = s_T;
  // every key equal to T is kept (always so when T is unique, the usual case for real-valued
  // scores): their order does not matter and nobody reads the per-row counts
  if (s_r == s_neq) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int u = blockIdx.x * 8 + warp;
  if (u >= NQB) return;
  const float* row = scores + (static_cast<size_t>(h) * NQB + u) * NKB;
  uint32_t n = 0;
  for (int v = lane; v < NKB; v += 32) n += (score_key(__ldg(row + v), force_diag && u == v) == T);
  for (int o = 16; o; o >>= 1) n += __shfl_xor_sync(0xFFFFFFFFu, n, o);
  if (lane == 0) row_ties[static_cast<size_t>(h) * NQB + u] = n;
}

// One warp per row: ties before this row (sum of row_ties of earlier rows), then 32 key blocks per
// step: keep = key > T, or key == T and its rank among the head's ties (flat-index order) < r.
__global__ void __launch_bounds__(256)
pack_write_kernel(const float* __restrict__ scores, int NQB, int NKB, int W, int force_diag,
                  const HeadState* __restrict__ state, const uint32_t* __restrict__ row_ties,
                  uint32_t* __restrict__ mask_bits) {
  const int h = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int u = blockIdx.x * 8 + warp;
  if (u >= NQB) return;
  const uint32_t T = state[h].prefix[4];
  const uint32_t r = state[h].k_rem[4];
  const bool all_equal_kept = r == state[h].n_equal;     // then keep = key >= T, no tie order needed
  uint32_t before = 0;
  if (!all_equal_kept) {
    for (int j = lane; j < u; j += 32) before += __ldg(row_ties + static_cast<size_t>(h) * NQB + j);
    for (int o = 16; o; o >>= 1) before += __shfl_xor_sync(0xFFFFFFFFu, before, o);
  }
  const float* row = scores + (static_cast<size_t>(h) * NQB + u) * NKB;
  uint32_t* out = mask_bits + (static_cast<size_t>(h) * NQB + u) * W;
  for (int w0 = 0; w0 < W; w0 += 4) {                     // four loads in flight per lane (L2 latency)
    float x[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int v = (w0 + q) * 32 + lane;
      x[q] = v < NKB ? __ldg(row + v) : 0.f;
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int w = w0 + q;
      if (w >= W) break;
      const int v = w * 32 + lane;
      const bool valid = v < NKB;
      const uint32_t key = valid ? score_key(x[q], force_diag && u == v) : 0u;
      uint32_t bits;
      if (all_equal_kept) {
        bits = __ballot_sync(0xFFFFFFFFu, valid && key >= T);
      } else {
        const uint32_t gt = __ballot_sync(0xFFFFFFFFu, valid && key > T);
        const uint32_t eq = __ballot_sync(0xFFFFFFFFu, valid && key == T);
        const uint32_t my_rank = before + __popc(eq & ((1u << lane) - 1u));
        bits = gt | __ballot_sync(0xFFFFFFFFu, valid && key == T && my_rank < r);
        before += __popc(eq);
      }
      if (lane == 0) out[w] = bits;
    }
  }
}

}  // namespace

size_t pack_mask_workspace_bytes(int H, int NQB, int NKB) {
  (void)NKB;
  return align256(static_cast<size_t>(H) * 4 * 256 * sizeof(uint32_t)) +
         align256(static_cast<size_t>(H) * sizeof(HeadState)) +
         align256(static_cast<size_t>(H) * NQB * sizeof(uint32_t));
}

cudaError_t launch_pack_mask(const float* scores, const float* density, uint32_t* mask_bits, int H,
                             int NQB, int NKB, int force_diag, void* ws, cudaStream_t st) {
  PackWs w = carve(ws, H, NQB);
  const int W = (NKB + 31) / 32;
  cudaError_t e = cudaMemsetAsync(w.hist, 0, static_cast<size_t>(H) * 4 * 256 * sizeof(uint32_t), st);
  if (e != cudaSuccess) return e;
  dim3 hgrid(static_cast<unsigned>((NQB + kHistRowsPerBlock - 1) / kHistRowsPerBlock), H);
  pack_hist_kernel<0><<<hgrid, kHistThreads, 0, st>>>(scores, density, NQB, NKB, force_diag, w.hist, w.state);
  pack_hist_kernel<1><<<hgrid, kHistThreads, 0, st>>>(scores, density, NQB, NKB, force_diag, w.hist, w.state);
  pack_hist_kernel<2><<<hgrid, kHistThreads, 0, st>>>(scores, density, NQB, NKB, force_diag, w.hist, w.state);
  pack_hist_kernel<3><<<hgrid, kHistThreads, 0, st>>>(scores, density, NQB, NKB, force_diag, w.hist, w.state);
  dim3 rgrid((NQB + 7) / 8, H);
  pack_row_ties_kernel<<<rgrid, 256, 0, st>>>(scores, density, NQB, NKB, force_diag, w.hist, w.state, w.row_ties);
  pack_write_kernel<<<rgrid, 256, 0, st>>>(scores, NQB, NKB, W, force_diag, w.state, w.row_ties, mask_bits);
  return cudaGetLastError();
}

}  // namespace sa

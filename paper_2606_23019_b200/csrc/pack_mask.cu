// pack_mask.cu -- sa_pack_mask: per-head top-fraction selection of block scores -> CRM bits.
//
// Mask instantiation M_p = 1(T <= p) (Sec. 4.1.2; Alg. 1 l.31) in the
// form BASELINE.json names: head h keeps the k_h best-scoring blocks of its NQB x NKB grid
// (readings P1-P4), written as CRM bit-rows (bit order PAPER.md:512,536).
//
// Exact selection without sorting: scores map to order-preserving uint32 keys; a radix select
// over three digits (11 + 11 + 10 bits) finds the k_h-th largest key T of the head (3 histogram
// passes over the scores, 56 MB at the 720p shape); keys > T are kept, and of the keys == T the
// first r in flat-index order, r = k_h - #(keys > T). Index order needs a prefix count of the
// ties: one per-row tie count pass, then each row's warp sums the rows before it and walks its
// own row 32 key blocks at a time with __ballot_sync, which is also what packs the bits. When all
// keys equal to T are kept (T unique: the usual case) both the tie counts and the prefix are skipped.
// Bandwidth/ALU work only; no tensor cores (HBM/L2-bound streaming, coalesced 128 B per warp).
#include "common.cuh"
#include <algorithm>

namespace sa {
namespace {

constexpr int kHistThreads = 256;
constexpr int kHistBlocksPerSm = 8;       // resident 256-thread histogram blocks per SM
constexpr long long kHistChunkMin = 4096; // fewest keys a histogram block takes
// the 32 key bits go in three digits from the top: 11 + 11 + 10
constexpr int kPasses = 3;
constexpr int kBins = 2048;               // bins of the widest digit
__host__ __device__ constexpr int digit_bits(int pass) { return pass < 2 ? 11 : 10; }
__host__ __device__ constexpr int digit_shift(int pass) { return pass == 0 ? 21 : pass == 1 ? 10 : 0; }

struct HeadState {      // per head, per pass p = 0..3: state after resolving passes < p
  uint32_t prefix[kPasses + 1];   // high bits fixed so far (prefix[p] has the digits of passes < p)
  uint32_t k_rem[kPasses + 1];    // how many keys with that prefix (ranked from the largest) still to take
  uint32_t n_equal;     // after the last pass: how many keys equal T = prefix[kPasses] the head holds
};

// workspace: hist uint32 [H][kPasses][kBins] | HeadState [H] | row_ties uint32 [H][NQB]
struct PackWs {
  uint32_t* hist;
  HeadState* state;
  uint32_t* row_ties;
};
__host__ __device__ inline size_t align256(size_t x) { return (x + 255) / 256 * 256; }
inline size_t hist_bytes(int H) { return static_cast<size_t>(H) * kPasses * kBins * sizeof(uint32_t); }

PackWs carve(void* ws, int H, int NQB) {
  char* p = static_cast<char*>(ws);
  PackWs w;
  w.hist = reinterpret_cast<uint32_t*>(p);
  p += align256(hist_bytes(H));
  w.state = reinterpret_cast<HeadState*>(p);
  p += align256(static_cast<size_t>(H) * sizeof(HeadState));
  w.row_ties = reinterpret_cast<uint32_t*>(p);
  (void)NQB;
  return w;
}

// fp32 score -> uint32 key, larger score <=> larger key. -0 is canonicalised to +0 (x + 0.0f);
// NaN sorts lowest (key 0); a forced diagonal entry takes the top key.
__device__ __forceinline__ uint32_t score_key(float x) {
  const float y = x + 0.0f;
  const uint32_t b = __float_as_uint(y);
  const uint32_t k = b ^ (static_cast<uint32_t>(static_cast<int32_t>(b) >> 31) | 0x80000000u);
  return x != x ? 0u : k;       // negative: ~b, positive: b | sign bit
}
__device__ __forceinline__ uint32_t score_key(float x, bool forced) {
  return forced ? 0xFFFFFFFFu : score_key(x);
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

// Resolve pass `pass - 1` from its histogram: find the digit whose bin holds the k_rem-th largest
// key, extend the prefix, reduce k_rem. Called by every block (256 threads; the head's bins are
// staged in `s_bins`, kBins words of shared memory the caller lends); the result lands in shared
// memory, and block 0 of the head records it for later kernels.
__device__ void resolve(int pass, int h, const float* density, int NQB, int NKB, int force_diag,
                        const uint32_t* hist, HeadState* state, uint32_t* s_bins,
                        uint32_t* s_prefix, uint32_t* s_krem, bool record,
                        uint32_t* s_nequal = nullptr) {
  __shared__ uint32_t s_warp[kHistThreads / 32];
  if (pass == 0) {
    if (threadIdx.x == 0) {
      *s_prefix = 0u;
      *s_krem = keep_count(density[h], NQB, NKB, force_diag);
      if (record) { state[h].prefix[0] = 0u; state[h].k_rem[0] = *s_krem; }
    }
    __syncthreads();
    return;
  }
  const int nb = 1 << digit_bits(pass - 1);
  const int per = nb / kHistThreads;                 // 8 or 4 bins per thread
  const uint32_t* hh = hist + (static_cast<size_t>(h) * kPasses + (pass - 1)) * kBins;
  const uint32_t prev_prefix = state[h].prefix[pass - 1];
  const uint32_t prev_krem = state[h].k_rem[pass - 1];
  for (int i = threadIdx.x; i < nb; i += kHistThreads) s_bins[i] = hh[i];
  __syncthreads();
  // bins from the largest digit down until the cumulative count reaches k_rem: thread t owns the
  // `per` bins nb-1-per*t downwards; a block scan gives the count above each thread's group
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  uint32_t c[8], sum = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    c[i] = i < per ? s_bins[nb - 1 - per * t - i] : 0u;
    sum += c[i];
  }
  uint32_t incl = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
    if (lane >= o) incl += v;
  }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  uint32_t warp_above = 0, all = 0;
#pragma unroll
  for (int w = 0; w < kHistThreads / 32; ++w) {
    const uint32_t v = s_warp[w];
    if (w < warp) warp_above += v;
    all += v;
  }
  incl += warp_above;
  uint32_t above = incl - sum;                         // keys in bins above this thread's group
  const bool here = above < prev_krem && incl >= prev_krem;
  // nobody reaches k_rem (cannot happen for a consistent histogram): fall to bin 0 like the walk
  const bool nobody = __syncthreads_or(here) == 0;
  if (here || (nobody && t == kHistThreads - 1)) {
    int bin = nb - 1 - per * t;
    for (int i = 0; i < per - 1; ++i, --bin) {
      if (above + c[i] >= prev_krem) break;
      above += c[i];
    }
    if (nobody) {                                      // walk semantics: stop at bin 0 whatever it holds
      bin = 0;
      above = all - s_bins[0];
    }
    *s_prefix = prev_prefix | (static_cast<uint32_t>(bin) << digit_shift(pass - 1));
    *s_krem = prev_krem - above;
    if (record) {
      state[h].prefix[pass] = *s_prefix;
      state[h].k_rem[pass] = *s_krem;
      if (pass == kPasses) state[h].n_equal = s_bins[bin];   // the bin of the full key
    }
    if (s_nequal) *s_nequal = s_bins[bin];
  }
  __syncthreads();
}

// Histogram of digit `PASS` (from the top) of the keys whose higher digits equal the prefix.
// A block takes `chunk` consecutive entries of one head's flat NQB x NKB array, four keys per
// 16-byte load (the few entries before / after the aligned part go one per thread); no row or
// column index is formed. The forced diagonal is a correction, not a per-key test: block 0 of the
// head takes the diagonal entries' real keys back out and counts the top key in their place
// (shared-memory counts wrap modulo 2^32; the global sum over the head's blocks is exact).
// Equal addresses of a warp's shared-memory increments merge in hardware (ATOMS.POPC.INC).
template <int PASS>
__global__ void __launch_bounds__(kHistThreads)
pack_hist_kernel(const float* __restrict__ scores, const float* __restrict__ density, int NQB,
                 int NKB, int force_diag, long long chunk, uint32_t* __restrict__ hist,
                 HeadState* state) {
  __shared__ uint32_t s_hist[kBins];
  __shared__ uint32_t s_prefix, s_krem;
  constexpr int nb = 1 << digit_bits(PASS);
  constexpr int shift = digit_shift(PASS);
  const int h = blockIdx.y;
  if (PASS > 0) griddep_wait();       // (launched programmatically behind the previous pass)
  resolve(PASS, h, density, NQB, NKB, force_diag, hist, state, s_hist, &s_prefix, &s_krem,
          blockIdx.x == 0);
  const uint32_t prefix = s_prefix;
  for (int i = threadIdx.x; i < nb; i += kHistThreads) s_hist[i] = 0u;
  __syncthreads();
  auto count = [&](uint32_t key, bool add) {
    if (PASS == 0 || ((key ^ prefix) >> (PASS == 0 ? 0 : shift + digit_bits(PASS))) == 0u) {
      if (add) atomicAdd(&s_hist[(key >> shift) & (nb - 1)], 1u);
      else atomicSub(&s_hist[(key >> shift) & (nb - 1)], 1u);
    }
  };
  const long long total = static_cast<long long>(NQB) * NKB;
  const long long c0 = static_cast<long long>(blockIdx.x) * chunk;
  const long long g0 = static_cast<long long>(h) * total + c0;           // index into `scores`
  const long long g1 = static_cast<long long>(h) * total + min(c0 + chunk, total);
  // 16-byte aligned part [ga, gb) of [g0, g1) (the pointer itself is only known to be a float's)
  const long long mis = static_cast<long long>((reinterpret_cast<uintptr_t>(scores) >> 2) & 3u);
  long long ga = ((g0 + mis + 3) & ~3LL) - mis;
  long long gb = ((g1 + mis) & ~3LL) - mis;
  if (ga > g1) ga = g1;
  if (gb < ga) gb = ga;
  if (threadIdx.x < ga - g0) count(score_key(__ldg(scores + g0 + threadIdx.x)), true);
  if (threadIdx.x < g1 - gb) count(score_key(__ldg(scores + gb + threadIdx.x)), true);
  const float4* vec = reinterpret_cast<const float4*>(scores + ga);
  const int nv = static_cast<int>((gb - ga) >> 2);                       // a chunk is < 2^31 keys
  for (int i0 = threadIdx.x; i0 < nv; i0 += 4 * kHistThreads) {          // four loads in flight
    float4 x[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int i = i0 + q * kHistThreads;
      x[q] = i < nv ? __ldg(vec + i) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      if (i0 + q * kHistThreads < nv) {
        count(score_key(x[q].x), true);
        count(score_key(x[q].y), true);
        count(score_key(x[q].z), true);
        count(score_key(x[q].w), true);
      }
    }
  }
  if (force_diag && blockIdx.x == 0) {
    const float* head = scores + static_cast<long long>(h) * total;
    const int nd = min(NQB, NKB);
    for (int u = threadIdx.x; u < nd; u += kHistThreads) {
      count(score_key(__ldg(head + static_cast<long long>(u) * (NKB + 1))), false);
      count(0xFFFFFFFFu, true);
    }
  }
  __syncthreads();
  uint32_t* hh = hist + (static_cast<size_t>(h) * kPasses + PASS) * kBins;
  for (int i = threadIdx.x; i < nb; i += kHistThreads)
    if (s_hist[i]) atomicAdd(hh + i, s_hist[i]);
}

// After the last pass: T = full key of the k_h-th largest, r = ties to keep. One warp per row counts the
// keys equal to T in its row. grid = (ceil(NQB / kTieRowsPerBlock), H), 8 warps per block.
constexpr int kTieRowsPerBlock = 64;
__global__ void __launch_bounds__(256)
pack_row_ties_kernel(const float* __restrict__ scores, const float* __restrict__ density, int NQB,
                     int NKB, int force_diag, const uint32_t* __restrict__ hist, HeadState* state,
                     uint32_t* __restrict__ row_ties) {
  __shared__ uint32_t s_bins[kBins];
  __shared__ uint32_t s_T, s_r, s_neq;
  const int h = blockIdx.y;
  griddep_wait();
  resolve(kPasses, h, density, NQB, NKB, force_diag, hist, state, s_bins, &s_T, &s_r,
          blockIdx.x == 0, &s_neq);
  const uint32_t T = s_T;
  // every key equal to T is kept (always so when T is unique, the usual case for real-valued
  // scores): their order does not matter and nobody reads the per-row counts
  if (s_r == s_neq) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int u_end = min((static_cast<int>(blockIdx.x) + 1) * kTieRowsPerBlock, NQB);
  for (int u = blockIdx.x * kTieRowsPerBlock + warp; u < u_end; u += 8) {
    const float* row = scores + (static_cast<size_t>(h) * NQB + u) * NKB;
    uint32_t n = 0;
    for (int v = lane; v < NKB; v += 32) n += (score_key(__ldg(row + v), force_diag && u == v) == T);
    for (int o = 16; o; o >>= 1) n += __shfl_xor_sync(0xFFFFFFFFu, n, o);
    if (lane == 0) row_ties[static_cast<size_t>(h) * NQB + u] = n;
  }
}

// One warp per row, 32 key blocks per step, __ballot_sync packs the bits. When every key equal to
// T is kept and T is the key of a number (the usual case), keep = score >= that number, compared
// as floats (NaN compares false = lowest, -0 equals +0: the key order), and the forced diagonal
// is one OR. Otherwise: ties before this row (sum of row_ties of earlier rows), keep = key > T,
// or key == T and its rank among the head's ties (flat-index order) < r.
__global__ void __launch_bounds__(256)
pack_write_kernel(const float* __restrict__ scores, int NQB, int NKB, int W, int force_diag,
                  const HeadState* __restrict__ state, const uint32_t* __restrict__ row_ties,
                  uint32_t* __restrict__ mask_bits) {
  const int h = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int u = blockIdx.x * 8 + warp;
  griddep_wait();
  if (u >= NQB) return;
  const uint32_t T = state[h].prefix[kPasses];
  const uint32_t r = state[h].k_rem[kPasses];
  const bool all_equal_kept = r == state[h].n_equal;     // then keep = key >= T, no tie order needed
  const float* row = scores + (static_cast<size_t>(h) * NQB + u) * NKB;
  uint32_t* out = mask_bits + (static_cast<size_t>(h) * NQB + u) * W;
  const float tf = __uint_as_float((T & 0x80000000u) ? (T ^ 0x80000000u) : ~T);   // key -> score
  if (all_equal_kept && tf == tf) {
    const int diag_w = (force_diag && u < NKB) ? (u >> 5) : -1;
    const uint32_t diag_bit = 1u << (u & 31);
    const int w_full = NKB >> 5;                          // words whose 32 key blocks all exist
    uint32_t mine = 0u;                                   // lane l holds word (w & ~31) + l
    int w = 0;
    for (; w + 4 <= w_full; w += 4) {                     // four loads in flight per lane
      float x[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) x[q] = __ldg(row + (w + q) * 32 + lane);
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        uint32_t bits = __ballot_sync(0xFFFFFFFFu, x[q] >= tf);
        if (w + q == diag_w) bits |= diag_bit;
        if (lane == ((w + q) & 31)) mine = bits;
      }
      if (((w + 4) & 31) == 0) out[w + 4 - 32 + lane] = mine;
    }
    for (; w < W; ++w) {
      const int v = w * 32 + lane;
      const float x = v < NKB ? __ldg(row + v) : 0.f;
      uint32_t bits = __ballot_sync(0xFFFFFFFFu, v < NKB && x >= tf);
      if (w == diag_w) bits |= diag_bit;
      if (lane == (w & 31)) mine = bits;
      if (((w + 1) & 31) == 0) out[w + 1 - 32 + lane] = mine;
    }
    if (lane < (W & 31)) out[(W & ~31) + lane] = mine;
    return;
  }
  uint32_t before = 0;
  if (!all_equal_kept) {
    for (int j = lane; j < u; j += 32) before += __ldg(row_ties + static_cast<size_t>(h) * NQB + j);
    for (int o = 16; o; o >>= 1) before += __shfl_xor_sync(0xFFFFFFFFu, before, o);
  }
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
  return align256(hist_bytes(H)) +
         align256(static_cast<size_t>(H) * sizeof(HeadState)) +
         align256(static_cast<size_t>(H) * NQB * sizeof(uint32_t));
}

cudaError_t launch_pack_mask(const float* scores, const float* density, uint32_t* mask_bits, int H,
                             int NQB, int NKB, int force_diag, void* ws, cudaStream_t st) {
  PackWs w = carve(ws, H, NQB);
  const int W = (NKB + 31) / 32;
  cudaError_t e = cudaMemsetAsync(w.hist, 0, hist_bytes(H), st);
  if (e != cudaSuccess) return e;
  // one wave of histogram blocks: each takes `chunk` consecutive keys of one head
  int n_sm = 0;
  e = device_sm_count(&n_sm);
  if (e != cudaSuccess) return e;
  const long long total = static_cast<long long>(NQB) * NKB;
  const long long per_head = std::max(1, n_sm * kHistBlocksPerSm / H);
  long long chunk = std::max(kHistChunkMin, (total + per_head - 1) / per_head);
  chunk = (chunk + 1023) / 1024 * 1024;
  dim3 hgrid(static_cast<unsigned>((total + chunk - 1) / chunk), H);
  pack_hist_kernel<0><<<hgrid, kHistThreads, 0, st>>>(scores, density, NQB, NKB, force_diag, chunk, w.hist, w.state);
  // the dependent kernels are launched programmatically: their launch overlaps the previous pass
  uint32_t* hist = w.hist;
  HeadState* state = w.state;
  const HeadState* cstate = w.state;
  const uint32_t* chist = w.hist;
  const uint32_t* cties = w.row_ties;
  if ((e = launch_pdl(pack_hist_kernel<1>, hgrid, dim3(kHistThreads), 0, st, scores, density, NQB, NKB, force_diag,
                      chunk, hist, state)) != cudaSuccess ||
      (e = launch_pdl(pack_hist_kernel<2>, hgrid, dim3(kHistThreads), 0, st, scores, density, NQB, NKB, force_diag,
                      chunk, hist, state)) != cudaSuccess)
    return e;
  dim3 tgrid((NQB + kTieRowsPerBlock - 1) / kTieRowsPerBlock, H);
  if ((e = launch_pdl(pack_row_ties_kernel, tgrid, dim3(256), 0, st, scores, density, NQB, NKB, force_diag, chist,
                      state, w.row_ties)) != cudaSuccess)
    return e;
  dim3 rgrid((NQB + 7) / 8, H);
  if ((e = launch_pdl(pack_write_kernel, rgrid, dim3(256), 0, st, scores, NQB, NKB, W, force_diag, cstate, cties,
                      mask_bits)) != cudaSuccess)
    return e;
  return cudaGetLastError();
}

}  // namespace sa

// west_update.cu -- sa_threshold_map_update: WEST's "Local Threshold Discovery" and "Topology
// Union" (Alg. 1 l.12-17) for a batch of calibration samples:
//     sort S and compute the cumulative sum C;  for each p in P find the cutoff tau s.t. C[tau] ~ p;
//     L(u,v) = min{p in P | block (u,v) is active at p};      T <- min(T, L).
// Readings P19-P20: descending sort with ties in flat-index order, C the inclusive
// cumulative sum divided by its total (a fraction of the head's attention mass), tau(p) the FIRST
// position with C[tau] >= p, a block active at no p keeps 1.0.
//
// Per (sample, head) segment, all kernels hand-written (no library sort or scan):
//   1. "Sort S": a stable least-significant-digit radix sort (4 passes of 8 bits) of the keys
//      ~(fp32 bits of S) with the flat index as payload. S >= 0, so the bit pattern orders like
//      the value and the complement turns the ascending radix order into DESCENDING S; the sort is
//      stable and the payload starts out ascending, so equal values stay in flat-index order --
//      the tie rule comes for free. A pass = per-tile digit histogram -> exclusive scan over
//      (digit, tile) -> stable scatter (warp-private running counters, match.any for the rank
//      inside a warp step). Pass 0 reads S itself, so no key buffer is built first.
//   2. "cumulative sum C ... cutoff": one CTA scans the sorted values in fp64 (warp-shuffle block
//      scan, chunk by chunk with a carry; twice: total, then levels); position r is active at p
//      exactly when r == 0 or C[r-1] / total < p, so L_r is the smallest level above C[r-1] / total;
//      it is merged into T[h] with an atomic min on the float's bit pattern (levels are positive,
//      so unsigned order = float order; min is order-independent, hence deterministic across the
//      samples that share a head).
// Streaming integer + fp64 ALU work, offline in the paper (Table 3).
#include "common.cuh"

namespace sa {
namespace {

constexpr int kScanThreads = 1024;
constexpr int kMaxLevels = 256;
constexpr int kSortThreads = 256;                 // 8 warps
constexpr int kPerThread = 16;
constexpr int kTile = kSortThreads * kPerThread;  // 4096 elements per block per pass
constexpr int kWarps = kSortThreads / 32;

__host__ __device__ inline size_t al256(size_t x) { return (x + 255) / 256 * 256; }

// descending-order key of a non-negative float (-0 -> +0 first)
__device__ __forceinline__ uint32_t desc_key(float s) { return ~__float_as_uint(s + 0.0f); }

// ---- pass step 1: digit histogram of one tile. hist[(seg * 256 + digit) * T + tile]
template <bool kFirst>
__global__ void __launch_bounds__(kSortThreads)
west_hist_kernel(const float* __restrict__ sig, const uint32_t* __restrict__ keys_in, int n, int T,
                 int shift, uint32_t* __restrict__ hist) {
  __shared__ uint32_t h[256];
  const int tile = blockIdx.x, seg = blockIdx.y, lane = threadIdx.x & 31;
  const size_t base = static_cast<size_t>(seg) * n;
  h[threadIdx.x] = 0u;
  __syncthreads();
#pragma unroll 4
  for (int i = 0; i < kPerThread; ++i) {
    const int e = tile * kTile + i * kSortThreads + threadIdx.x;
    const bool valid = e < n;
    uint32_t key = 0u;
    if (valid) key = kFirst ? desc_key(__ldg(sig + base + e)) : __ldg(keys_in + base + e);
    // lanes with the same digit add once (the top byte of a float is shared by most of a warp)
    const uint32_t d = valid ? ((key >> shift) & 255u) : (256u + lane);
    const uint32_t peers = __match_any_sync(0xFFFFFFFFu, d);
    if (valid && (peers & ((1u << lane) - 1u)) == 0u) atomicAdd(&h[d], __popc(peers));
  }
  __syncthreads();
  hist[(static_cast<size_t>(seg) * 256 + threadIdx.x) * T + tile] = h[threadIdx.x];
}

// warp-shuffle block scan (exclusive) of one value per thread; `total` = sum over the block.
// tmp: shared, blockDim / 32 + 1 entries. All threads must call it.
template <typename V>
__device__ __forceinline__ V block_exclusive_scan(V v, V* tmp, V& total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  V inc = v;
#pragma unroll
  for (int s = 1; s < 32; s <<= 1) {
    const V o = __shfl_up_sync(0xFFFFFFFFu, inc, s);
    if (lane >= s) inc += o;
  }
  if (lane == 31) tmp[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    const V w = lane < nw ? tmp[lane] : V(0);
    V winc = w;
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
      const V o = __shfl_up_sync(0xFFFFFFFFu, winc, s);
      if (lane >= s) winc += o;
    }
    if (lane < nw) tmp[lane] = winc - w;            // exclusive prefix of the warp totals
    if (lane == 31) tmp[nw] = winc;                 // block total
  }
  __syncthreads();
  const V res = inc - v + tmp[warp];
  total = tmp[nw];
  __syncthreads();                                  // tmp is reused by the caller's next chunk
  return res;
}

// ---- pass step 2: exclusive scan of a segment's (digit, tile) counts, in place
__global__ void __launch_bounds__(kScanThreads)
west_offsets_kernel(uint32_t* __restrict__ hist, int T) {
  __shared__ uint32_t tmp[kScanThreads / 32 + 1];
  uint32_t* h = hist + static_cast<size_t>(blockIdx.x) * 256 * T;
  const int len = 256 * T;
  uint32_t carry = 0u;
  for (int base = 0; base < len; base += kScanThreads) {
    const int i = base + threadIdx.x;
    const uint32_t v = i < len ? h[i] : 0u;
    uint32_t chunk;
    const uint32_t ex = block_exclusive_scan(v, tmp, chunk);
    if (i < len) h[i] = carry + ex;
    carry += chunk;
  }
}

// ---- pass step 3: stable scatter of one tile. Warp w owns elements [512 w, 512 w + 512) of the
// tile and walks them in 16 steps of 32 consecutive elements; cnt[w][d] counts the digit-d elements
// the warp has passed, so an element's rank among the tile's digit-d elements is (digit-d elements
// of lower warps) + cnt[w][d] at its step + (lower lanes with the same digit in its step).
template <bool kFirst>
__global__ void __launch_bounds__(kSortThreads)
west_scatter_kernel(const float* __restrict__ sig, const uint32_t* __restrict__ keys_in,
                    const uint32_t* __restrict__ idx_in, int n, int T, int shift,
                    const uint32_t* __restrict__ offsets, uint32_t* __restrict__ keys_out,
                    uint32_t* __restrict__ idx_out) {
  __shared__ uint32_t cnt[kWarps][256];
  __shared__ uint32_t gbase[256];
  const int tile = blockIdx.x, seg = blockIdx.y;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const size_t base = static_cast<size_t>(seg) * n;
  for (int w = 0; w < kWarps; ++w) cnt[w][threadIdx.x] = 0u;
  gbase[threadIdx.x] = offsets[(static_cast<size_t>(seg) * 256 + threadIdx.x) * T + tile];
  __syncthreads();
  uint32_t key[kPerThread], idx[kPerThread];
  uint16_t rank[kPerThread];
#pragma unroll
  for (int s = 0; s < kPerThread; ++s) {
    const int e = tile * kTile + warp * (32 * kPerThread) + s * 32 + lane;
    const bool valid = e < n;
    key[s] = 0u;
    idx[s] = static_cast<uint32_t>(e);
    if (valid) {
      key[s] = kFirst ? desc_key(__ldg(sig + base + e)) : __ldg(keys_in + base + e);
      if (!kFirst) idx[s] = __ldg(idx_in + base + e);
    }
    const uint32_t d = valid ? ((key[s] >> shift) & 255u) : (256u + lane);
    const uint32_t peers = __match_any_sync(0xFFFFFFFFu, d);
    const uint32_t below = __popc(peers & ((1u << lane) - 1u));
    uint32_t r = 0u;
    if (valid) r = cnt[warp][d] + below;
    __syncwarp();
    if (valid && below == 0u) cnt[warp][d] += __popc(peers);
    __syncwarp();
    rank[s] = static_cast<uint16_t>(r);
  }
  __syncthreads();
  {                                               // exclusive prefix over the warps, per digit
    uint32_t run = 0u;
    for (int w = 0; w < kWarps; ++w) {
      const uint32_t c = cnt[w][threadIdx.x];
      cnt[w][threadIdx.x] = run;
      run += c;
    }
  }
  __syncthreads();
#pragma unroll
  for (int s = 0; s < kPerThread; ++s) {
    const int e = tile * kTile + warp * (32 * kPerThread) + s * 32 + lane;
    if (e < n) {
      const uint32_t d = (key[s] >> shift) & 255u;
      const size_t pos = base + gbase[d] + cnt[warp][d] + rank[s];
      keys_out[pos] = key[s];
      idx_out[pos] = idx[s];
    }
  }
}

// ---- cumulative sum, per-level cutoffs, local map, topology union
__global__ void __launch_bounds__(kScanThreads)
west_scan_kernel(const uint32_t* __restrict__ sorted_keys, const uint32_t* __restrict__ sorted_idx,
                 const float* __restrict__ levels, int n_levels, float* __restrict__ tmap, int H, int n) {
  __shared__ double tmp[kScanThreads / 32 + 1];
  __shared__ float lv[kMaxLevels];
  const int seg = blockIdx.x, h = seg % H;
  const uint32_t* keys = sorted_keys + static_cast<size_t>(seg) * n;
  const uint32_t* idxs = sorted_idx + static_cast<size_t>(seg) * n;
  unsigned* T = reinterpret_cast<unsigned*>(tmap + static_cast<size_t>(h) * n);
  for (int i = threadIdx.x; i < n_levels; i += kScanThreads) lv[i] = levels[i];
  __syncthreads();
  double total = 0.0;
  // pass 0 finds the total (the last inclusive prefix), pass 1 redoes the identical scan and uses
  // the exclusive prefix C[r-1] of every position
  for (int pass = 0; pass < 2; ++pass) {
    double carry = 0.0;                         // inclusive prefix of everything before this chunk
    for (int base = 0; base < n; base += kScanThreads) {
      const int r = base + threadIdx.x;
      const double val = r < n ? static_cast<double>(__uint_as_float(~keys[r])) : 0.0;
      double chunk;
      const double excl = block_exclusive_scan(val, tmp, chunk);
      if (pass == 1 && r < n) {
        float L = 1.0f;                         // active at no level: the map's initial max value
        if (r == 0) {
          L = lv[0];
        } else {
          const double cn = (carry + excl) / total;          // C[r-1] / C[last]
          int lo = 0, hi = n_levels;                         // first level with lv > cn
          while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (static_cast<double>(lv[mid]) > cn) hi = mid; else lo = mid + 1;
          }
          if (lo < n_levels) L = lv[lo];
        }
        atomicMin(T + idxs[r], __float_as_uint(L));
      }
      carry += chunk;
    }
    total = carry;
  }
}

struct SortBuffers {
  uint32_t *keys[2], *idx[2], *hist;
};
SortBuffers carve(void* ws, size_t total, size_t n_seg, int T) {
  char* p = static_cast<char*>(ws);
  SortBuffers b;
  for (int i = 0; i < 2; ++i) { b.keys[i] = reinterpret_cast<uint32_t*>(p); p += al256(total * 4); }
  for (int i = 0; i < 2; ++i) { b.idx[i] = reinterpret_cast<uint32_t*>(p); p += al256(total * 4); }
  b.hist = reinterpret_cast<uint32_t*>(p);
  (void)n_seg; (void)T;
  return b;
}

}  // namespace

size_t threshold_update_workspace_bytes(int B, int H, int NQB, int NKB) {
  const size_t n_seg = static_cast<size_t>(B) * H, n = static_cast<size_t>(NQB) * NKB;
  const size_t T = (n + kTile - 1) / kTile;
  return 4 * al256(n_seg * n * 4) + al256(n_seg * 256 * T * 4);
}

cudaError_t launch_threshold_update(const float* sig, const float* levels, int n_levels, float* tmap,
                                    int B, int H, int NQB, int NKB, void* ws, cudaStream_t st,
                                    int* n_launch) {
  const int n_seg = B * H, n = NQB * NKB;
  const int T = (n + kTile - 1) / kTile;
  const SortBuffers b = carve(ws, static_cast<size_t>(n_seg) * n, n_seg, T);
  const dim3 grid(T, n_seg);
  int src = 0;
  for (int pass = 0; pass < 4; ++pass) {
    const int shift = 8 * pass;
    if (pass == 0) west_hist_kernel<true><<<grid, kSortThreads, 0, st>>>(sig, nullptr, n, T, shift, b.hist);
    else west_hist_kernel<false><<<grid, kSortThreads, 0, st>>>(nullptr, b.keys[src], n, T, shift, b.hist);
    west_offsets_kernel<<<n_seg, kScanThreads, 0, st>>>(b.hist, T);
    if (pass == 0)
      west_scatter_kernel<true><<<grid, kSortThreads, 0, st>>>(sig, nullptr, nullptr, n, T, shift, b.hist,
                                                                b.keys[0], b.idx[0]);
    else
      west_scatter_kernel<false><<<grid, kSortThreads, 0, st>>>(nullptr, b.keys[src], b.idx[src], n, T, shift,
                                                                 b.hist, b.keys[src ^ 1], b.idx[src ^ 1]);
    if (pass > 0) src ^= 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  west_scan_kernel<<<n_seg, kScanThreads, 0, st>>>(b.keys[src], b.idx[src], levels, n_levels, tmap, H, n);
  *n_launch += 13;
  return cudaGetLastError();
}

}  // namespace sa

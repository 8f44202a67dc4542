// west_update.cu -- sa_threshold_map_update: WEST's "Local Threshold Discovery" and "Topology
// Union" (Alg. 1 l.12-17) for a batch of calibration samples:
//     sort S and compute the cumulative sum C;  for each p in P find the cutoff tau s.t. C[tau] ~ p;
//     L(u,v) = min{p in P | block (u,v) is active at p};      T <- min(T, L).
// Readings P19-P20: descending sort with ties in flat-index order, C the inclusive
// cumulative sum divided by its total (a fraction of the head's attention mass), tau(p) the FIRST
// position with C[tau] >= p, a block active at no p keeps 1.0.
//
// Per (sample, head) segment:
//   1. 64-bit keys  (fp32 bits of S) << 32 | ~flat index : one descending key sort gives the order
//      AND the tie rule, whatever the sort's stability (S >= 0, so the bit pattern orders like the
//      value). The sort is a library primitive (cub::DeviceSegmentedRadixSort).
//   2. one CTA scans the sorted values in fp64 (block scan, chunk by chunk with a carry); position r
//      is active at p exactly when r == 0 or C[r-1] / total < p, so L_r is the smallest level above
//      C[r-1] / total; it is merged into T[h] with an atomic min on the float's bit pattern
//      (levels are positive, so unsigned order = float order; min is order-independent, hence
//      deterministic across the samples that share a head).
// Streaming/sort-bound integer + fp64 ALU work, offline in the paper (Table 3).
#include <cub/cub.cuh>

#include "common.cuh"

namespace sa {
namespace {

constexpr int kThreads = 1024;
constexpr int kMaxLevels = 256;

__host__ __device__ inline size_t al256(size_t x) { return (x + 255) / 256 * 256; }

__global__ void west_keys_kernel(const float* __restrict__ sig, unsigned long long* __restrict__ keys,
                                 int* __restrict__ offsets, int n_seg, int n) {
  const long long total = static_cast<long long>(n_seg) * n;
  const long long stride = static_cast<long long>(gridDim.x) * blockDim.x;
  const long long first = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  for (long long i = first; i <= n_seg; i += stride) offsets[i] = static_cast<int>(i * n);   // segment offsets
  for (long long i = first; i < total; i += stride) {
    const unsigned idx = static_cast<unsigned>(i % n);
    const float s = sig[i] + 0.0f;                                  // -0 -> +0
    keys[i] = (static_cast<unsigned long long>(__float_as_uint(s)) << 32) | (0xFFFFFFFFu - idx);
  }
}

__global__ void __launch_bounds__(kThreads)
west_scan_kernel(const unsigned long long* __restrict__ sorted, const float* __restrict__ levels,
                 int n_levels, float* __restrict__ tmap, int H, int n) {
  using BlockScan = cub::BlockScan<double, kThreads>;
  __shared__ typename BlockScan::TempStorage tmp;
  __shared__ float lv[kMaxLevels];
  const int seg = blockIdx.x, h = seg % H;
  const unsigned long long* keys = sorted + static_cast<size_t>(seg) * n;
  unsigned* T = reinterpret_cast<unsigned*>(tmap + static_cast<size_t>(h) * n);
  for (int i = threadIdx.x; i < n_levels; i += kThreads) lv[i] = levels[i];
  __syncthreads();
  double total = 0.0;
  // pass 0 finds the total (the last inclusive prefix), pass 1 redoes the identical scan and uses
  // the exclusive prefix C[r-1] of every position
  for (int pass = 0; pass < 2; ++pass) {
    double carry = 0.0;                         // inclusive prefix of everything before this chunk
    for (int base = 0; base < n; base += kThreads) {
      const int r = base + threadIdx.x;
      const unsigned long long key = r < n ? keys[r] : 0ull;
      const double val =
          r < n ? static_cast<double>(__uint_as_float(static_cast<unsigned>(key >> 32))) : 0.0;
      double excl, chunk;
      BlockScan(tmp).ExclusiveSum(val, excl, chunk);
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
        const unsigned idx = 0xFFFFFFFFu - static_cast<unsigned>(key & 0xFFFFFFFFull);
        atomicMin(T + idx, __float_as_uint(L));
      }
      carry += chunk;
      __syncthreads();                          // TempStorage is reused by the next chunk
    }
    total = carry;
  }
}

}  // namespace

size_t threshold_update_workspace_bytes(int B, int H, int NQB, int NKB) {
  const size_t n_seg = static_cast<size_t>(B) * H, n = static_cast<size_t>(NQB) * NKB;
  size_t temp = 0;
  cub::DeviceSegmentedRadixSort::SortKeysDescending(
      nullptr, temp, static_cast<const unsigned long long*>(nullptr),
      static_cast<unsigned long long*>(nullptr), static_cast<int>(n_seg * n), static_cast<int>(n_seg),
      static_cast<const int*>(nullptr), static_cast<const int*>(nullptr));
  return 2 * al256(n_seg * n * 8) + al256((n_seg + 1) * 4) + al256(temp);
}

cudaError_t launch_threshold_update(const float* sig, const float* levels, int n_levels, float* tmap,
                                    int B, int H, int NQB, int NKB, void* ws, cudaStream_t st,
                                    int* n_launch) {
  const int n_seg = B * H, n = NQB * NKB;
  char* p = static_cast<char*>(ws);
  unsigned long long* keys_in = reinterpret_cast<unsigned long long*>(p);
  p += al256(static_cast<size_t>(n_seg) * n * 8);
  unsigned long long* keys_out = reinterpret_cast<unsigned long long*>(p);
  p += al256(static_cast<size_t>(n_seg) * n * 8);
  int* offsets = reinterpret_cast<int*>(p);
  p += al256((static_cast<size_t>(n_seg) + 1) * 4);
  size_t temp = 0;
  cub::DeviceSegmentedRadixSort::SortKeysDescending(nullptr, temp, keys_in, keys_out, n_seg * n, n_seg,
                                                    offsets, offsets + 1);
  const long long total = static_cast<long long>(n_seg) * n;
  long long blocks = (total + 255) / 256;
  if (blocks > 148 * 32) blocks = 148 * 32;
  west_keys_kernel<<<static_cast<unsigned>(blocks), 256, 0, st>>>(sig, keys_in, offsets, n_seg, n);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  e = cub::DeviceSegmentedRadixSort::SortKeysDescending(p, temp, keys_in, keys_out, n_seg * n, n_seg,
                                                        offsets, offsets + 1, 0, 64, st);
  if (e != cudaSuccess) return e;
  west_scan_kernel<<<n_seg, kThreads, 0, st>>>(keys_out, levels, n_levels, tmap, H, n);
  *n_launch += 2;    // + the library sort's own launches
  return cudaGetLastError();
}

}  // namespace sa

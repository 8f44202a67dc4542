// schedule.cu -- work assignment pre-pass (DESIGN.md step A1) and the CRM walk test kernel.
//
// One unit of work is (batch, head, query block) (the CRM iterator replaces the
// dense KV-block iterator of FlashAttention, whose forward pass gives one thread block one query
// block). The paper is silent on load balance; per-row popcounts are uneven (edge blocks, sinks,
// per-head density), so the pre-pass orders the work: (b,h) groups heaviest first (keeps the
// concurrently running CTAs on one or two heads, whose K/V then stay in L2) and, inside a group,
// items by descending cost (longest-processing-time first; the tail is the lightest rows of the
// lightest head). Everything here is integer work on the packed mask only.
#include "common.cuh"

namespace sa {

size_t fwd_workspace_bytes(int B, int H, int NQB) {
  const size_t BH = static_cast<size_t>(B) * H;
  const size_t n = 16 + 3 * BH + 2 * BH * static_cast<size_t>(NQB);
  return ((n * sizeof(int32_t) + 255) / 256) * 256;
}

FwdWorkspace carve_fwd_workspace(void* ws, int B, int H, int NQB) {
  const size_t BH = static_cast<size_t>(B) * H;
  int32_t* p = static_cast<int32_t*>(ws);
  FwdWorkspace w;
  w.cursor = p;
  w.head_cost = p + 16;
  w.head_order = w.head_cost + BH;
  w.kmax2 = reinterpret_cast<float*>(w.head_order + BH);
  w.local_order = w.head_order + 2 * BH;
  w.unit_order = w.local_order + BH * static_cast<size_t>(NQB);
  return w;
}

namespace {

constexpr int kSortThreads = 1024;

// grid = B*H blocks. Item i of group (b,h) covers query blocks [i*rpi, min((i+1)*rpi, NQB)); its
// cost is the number of active (query block, key block) tiles in it. local_order[bh][pos] = item
// with the pos-th largest cost (ties: lower item first).
__global__ void __launch_bounds__(kSortThreads)
schedule_sort_kernel(const uint32_t* __restrict__ mask_bits, int H, int NQB, int NKB, int W,
                     int rpi, int items, int32_t* __restrict__ head_cost,
                     int32_t* __restrict__ local_order, float* __restrict__ kmax2) {
  extern __shared__ int32_t s_cost[];
  __shared__ int s_total;
  const int bh = blockIdx.x;
  const int h = bh % H;
  if (threadIdx.x == 0) {
    s_total = 0;
    kmax2[bh] = 0.f;                 // key_norm_kernel (next on the stream) takes the max into it
  }
  __syncthreads();
  const uint32_t tail_mask = (NKB & 31) ? ((1u << (NKB & 31)) - 1u) : 0xFFFFFFFFu;
  int my_total = 0;
  for (int i = threadIdx.x; i < items; i += blockDim.x) {
    int c = 0;
    for (int r = i * rpi; r < min((i + 1) * rpi, NQB); ++r) {
      const uint32_t* row = mask_bits + (static_cast<size_t>(h) * NQB + r) * W;
      for (int w = 0; w < W; ++w) {
        uint32_t x = __ldg(row + w);
        if (w == W - 1) x &= tail_mask;
        c += __popc(x);
      }
    }
    s_cost[i] = c;
    my_total += c;
  }
  atomicAdd(&s_total, my_total);
  __syncthreads();
  if (threadIdx.x == 0) head_cost[bh] = s_total;
  for (int i = threadIdx.x; i < items; i += blockDim.x) {
    const int ci = s_cost[i];
    int pos = 0;
    for (int j = 0; j < items; ++j) {
      const int cj = s_cost[j];
      pos += (cj > ci) || (cj == ci && j < i);
    }
    local_order[static_cast<size_t>(bh) * items + pos] = i;
  }
}

// unit_order[p] = global item id (bh * items + local item) issued p-th; resets the cursor.
// Every block first ranks the (b,h) groups by (cost descending, id ascending) into shared memory.
__global__ void __launch_bounds__(256)
schedule_flatten_kernel(const int32_t* __restrict__ head_cost, int32_t* __restrict__ head_order,
                        const int32_t* __restrict__ local_order, int BH, int items,
                        int32_t* __restrict__ unit_order, int32_t* __restrict__ cursor) {
  extern __shared__ int32_t s_order[];
  for (int g = threadIdx.x; g < BH; g += blockDim.x) {
    const int cg = __ldg(head_cost + g);
    int ahead = 0;
    for (int j = 0; j < BH; ++j) {
      const int cj = __ldg(head_cost + j);
      ahead += (cj > cg) || (cj == cg && j < g);
    }
    s_order[ahead] = g;
  }
  __syncthreads();
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p == 0) *cursor = 0;
  if (p >= BH * items) return;
  const int rank = p / items, pos = p % items;
  const int bh = s_order[rank];
  if (pos == 0) head_order[rank] = bh;
  unit_order[p] = bh * items + local_order[static_cast<size_t>(bh) * items + pos];
}

// kmax2[bh] = max over the valid keys j of |k_j|^2 (D = 128). Half a warp per key row: 16 lanes x 16
// bytes = one 256 B row per load, fully coalesced; 4 shuffles fold the 16 partial sums.
// The forward kernel turns it into the Cauchy-Schwarz bound scale * |q_i| * max_j |k_j| >= every
// score of query row i, which lets it fix the softmax reference point of a row for a whole item.
constexpr int kNormThreads = 256;
constexpr int kNormRowsPerBlock = 1024;
__global__ void __launch_bounds__(kNormThreads)
key_norm_kernel(const __nv_bfloat16* __restrict__ k, int N, int n_valid, float* __restrict__ kmax2) {
  const int bh = blockIdx.y;
  const int r0 = blockIdx.x * kNormRowsPerBlock;
  const int r1 = min(r0 + kNormRowsPerBlock, n_valid);
  const int half = threadIdx.x >> 4, sub = threadIdx.x & 15;       // 16 half-warps per block
  const uint4* base = reinterpret_cast<const uint4*>(k + static_cast<size_t>(bh) * N * 128);
  float best = 0.f;
#pragma unroll 4
  for (int rb = r0; rb < r1; rb += kNormThreads / 16) {       // uniform trip count (shuffles inside)
    const int r = rb + half;
    const uint4 x = r < r1 ? __ldg(base + static_cast<size_t>(r) * 16 + sub) : make_uint4(0u, 0u, 0u, 0u);
    const uint32_t w[4] = {x.x, x.y, x.z, x.w};
    float acc = 0.f;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float lo = __uint_as_float(w[i] << 16), hi = __uint_as_float(w[i] & 0xFFFF0000u);
      acc = fmaf(lo, lo, acc);
      acc = fmaf(hi, hi, acc);
    }
#pragma unroll
    for (int s = 8; s > 0; s >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, s);
    best = fmaxf(best, acc);
  }
  best = fmaxf(best, __shfl_xor_sync(0xFFFFFFFFu, best, 16));
  if ((threadIdx.x & 31) == 0)
    atomicMax(reinterpret_cast<unsigned*>(kmax2 + bh), __float_as_uint(best));   // non-negative floats
}

__global__ void __launch_bounds__(128)
enumerate_kernel(const uint32_t* __restrict__ mask_bits, int rows, int NKB, int W,
                 int32_t* __restrict__ idx, int32_t* __restrict__ cnt) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= rows) return;
  CrmIter it;
  it.init(mask_bits + static_cast<size_t>(r) * W, W, NKB);
  int n = 0;
  for (int v = it.index(); v >= 0; it.next(), v = it.index())
    idx[static_cast<size_t>(r) * NKB + n++] = v;
  cnt[r] = n;
}

}  // namespace

cudaError_t launch_schedule(const FwdParams& p, const FwdWorkspace& w, int rpi, cudaStream_t st,
                            int* n_launch, bool reuse) {
  const int BH = p.B * p.H;
  const int items = (p.NQB + rpi - 1) / rpi;
  if (reuse) {
    // the work list in the workspace is still valid (same mask): only reset what a call consumes
    cudaError_t e = cudaMemsetAsync(w.cursor, 0, sizeof(int32_t), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(w.kmax2, 0, static_cast<size_t>(BH) * sizeof(float), st);
    if (e != cudaSuccess) return e;
  } else {
  schedule_sort_kernel<<<BH, kSortThreads, items * sizeof(int32_t), st>>>(
      p.mask_bits, p.H, p.NQB, p.NKB, p.W, rpi, items, w.head_cost, w.local_order, w.kmax2);
  const int total = BH * items;
  schedule_flatten_kernel<<<(total + 255) / 256, 256, BH * sizeof(int32_t), st>>>(
      w.head_cost, w.head_order, w.local_order, BH, items, w.unit_order, w.cursor);
  *n_launch += 2;
  }
  if (p.D == 128 && p.kmax2 != nullptr) {   // the tcgen05 kernel's score bound needs max |k|^2
    const dim3 grid((p.n_valid + kNormRowsPerBlock - 1) / kNormRowsPerBlock, BH);
    key_norm_kernel<<<grid, kNormThreads, 0, st>>>(p.k, p.N, p.n_valid, w.kmax2);
    *n_launch += 1;
  }
  return cudaGetLastError();
}

cudaError_t launch_enumerate(const uint32_t* mask_bits, int H, int NQB, int NKB, int32_t* idx,
                             int32_t* cnt, cudaStream_t st) {
  const int rows = H * NQB;
  const int W = (NKB + 31) / 32;
  enumerate_kernel<<<(rows + 127) / 128, 128, 0, st>>>(mask_bits, rows, NKB, W, idx, cnt);
  return cudaGetLastError();
}

}  // namespace sa

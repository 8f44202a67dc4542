// schedule.cu -- work assignment pre-pass (DESIGN.md step A1) and the CRM walk test kernel.
//
// One unit of work is (batch, head, query block) (the CRM iterator replaces the
// dense KV-block iterator of FlashAttention, whose forward pass gives one thread block one query
// block). The paper is silent on load balance; per-row popcounts are uneven (edge blocks, sinks,
// per-head density). The pre-pass builds the work items and orders them:
//   * an item is one query block or, for the tcgen05 kernel on large problems, a PAIR of query
//     blocks of one (batch, head) that share every staged K/V tile. Adjacent blocks (2i, 2i+1)
//     are paired when their popcounts are balanced (3D-local masks make neighbours share most key
//     blocks). A block that is much heavier than its neighbour would run alone for most of the
//     item (one softmax warpgroup idle), so both go to a pool instead; the pool is sorted by
//     popcount and matched within windows of four rows by bit-row overlap (__popc(row_a & row_b)):
//     heavy rows meet heavy rows (BASELINE.json's adversarial case: the fully dense rows pair up),
//     and among equally heavy candidates the partner with the most shared key blocks wins.
//   * (b,h) groups heaviest first (keeps the concurrently running CTAs on one or two heads, whose
//     K/V then stay in L2) and, inside a group, items by descending cost (longest-processing-time
//     first; the tail is the lightest items of the lightest head).
//   * when the pairs do not fill a whole number of rounds over the SMs and there are few rounds
//     (fwd_tail_plan), the lightest items of every group -- as many in total as the last round
//     holds -- are issued in 2 or 4 PARTS each: the same rows over consecutive key ranges that
//     hold equal shares of the item's key blocks, at the very end of the order, so that the last
//     round is a half or a quarter as long. A part leaves its normalised O and its lse in a
//     scratch slot; combine_parts_kernel merges the parts of a row (a fixed order: deterministic).
// Everything here is integer work on the packed mask only; the resulting order cannot change any
// output bit (each query block is reduced by one CTA over its key blocks in ascending order).
#include "common.cuh"

namespace sa {

// a part's fixed cost is ~4 key blocks' worth: no shorter parts than this (measured: parts of 16-25
// key blocks lose 1-2% at density 0.05-0.1)
constexpr int kMinPartBlocks = 32;

// Pairs that do not fill a whole number of rounds over the SMs: with few rounds the partly filled
// last one is a large share of the launch (N = 16384, H = 12: 768 pairs = 5 rounds of 148 + 28 pairs,
// the sixth round as long as the others). Its pairs are issued in 2 or 4 parts (key ranges with the
// same share of the pair's key blocks), whichever makes ceil(rem * parts / n_sm) / parts, the length of
// that round in units of a pair, smallest; combine_parts_kernel merges a row's parts afterwards.
TailPlan fwd_tail_plan(int B, int H, int NQB, int NKB, int n_sm) {
  TailPlan t;
  const long long groups = static_cast<long long>(B) * H;
  const long long n_pairs = groups * ((NQB + 1) / 2);
  if (n_sm <= 0 || n_pairs < 2LL * n_sm || NKB > 0xFFFF) return t;
  const int max_parts = NKB / kMinPartBlocks;                 // a dense row's key blocks allow this many parts
  const long long rounds = n_pairs / n_sm, rem = n_pairs % n_sm;
  if (rem == 0) return t;
  long long best_num = 1, best_den = 1;                       // length of the last round: num / den
  for (int parts = 2; parts <= 4 && parts <= max_parts; parts *= 2) {
    const long long num = (rem * parts + n_sm - 1) / n_sm;    // rounds of 1/parts each
    if (num * best_den < best_num * parts) {
      best_num = num;
      best_den = parts;
      t.parts = parts;
    }
  }
  // worth it from 3% of the launch on (the parts cost a fourth launch and ~4 key blocks' time each)
  if (t.parts && (best_den - best_num) * 100 < 3 * best_den * (rounds + 1)) t.parts = 0;
  if (t.parts) t.rem = static_cast<int>(rem);
  return t;
}

static size_t al256(size_t x) { return (x + 255) / 256 * 256; }

size_t fwd_workspace_bytes(int B, int H, int NQB, int W, TailPlan plan) {
  const size_t BH = static_cast<size_t>(B) * H;
  // two int4 arrays of BH*NQB records (+ alignment), then the parts' task list and results
  const size_t words = 20 + 4 * BH + 8 * BH * static_cast<size_t>(NQB);
  const size_t slots = static_cast<size_t>(plan.rem) * plan.parts;
  return al256(words * sizeof(int32_t)) + al256(static_cast<size_t>(plan.rem) * sizeof(int4)) +
         al256(slots * 2 * W * sizeof(uint32_t)) +
         al256(slots * 2 * 128 * 128 * sizeof(__nv_bfloat16)) + al256(slots * 2 * 128 * sizeof(float));
}

FwdWorkspace carve_fwd_workspace(void* ws, int B, int H, int NQB, int W, TailPlan plan) {
  const size_t BH = static_cast<size_t>(B) * H;
  int32_t* p = static_cast<int32_t*>(ws);
  FwdWorkspace w;
  w.cursor = p;
  w.n_items = p + 1;
  w.stats = p + 2;
  w.head_cost = p + 16;
  w.head_count = w.head_cost + BH;
  w.head_tail = w.head_count + BH;
  w.kmax2 = reinterpret_cast<float*>(w.head_tail + BH);
  int32_t* rec = w.head_tail + 2 * BH;
  rec += (4 - ((rec - p) & 3)) & 3;                                       // int4 alignment (ws is 16 B aligned)
  w.local_items = reinterpret_cast<int4*>(rec);
  w.items = w.local_items + BH * static_cast<size_t>(NQB);
  const size_t words = 20 + 4 * BH + 8 * BH * static_cast<size_t>(NQB);
  char* c = static_cast<char*>(ws) + al256(words * sizeof(int32_t));
  const size_t slots = static_cast<size_t>(plan.rem) * plan.parts;
  w.tasks = reinterpret_cast<int4*>(c);
  c += al256(static_cast<size_t>(plan.rem) * sizeof(int4));
  w.part_mask = reinterpret_cast<uint32_t*>(c);
  c += al256(slots * 2 * W * sizeof(uint32_t));
  w.part_out = reinterpret_cast<__nv_bfloat16*>(c);
  c += al256(slots * 2 * 128 * 128 * sizeof(__nv_bfloat16));
  w.part_lse = reinterpret_cast<float*>(c);
  return w;
}

namespace {

constexpr int kSortThreads = 1024;
constexpr int kMinSingleBlocks = 3;       // rows of a tail pair that run as single-row items hold at least this many
constexpr int kMaxTail = 128;             // rows-in-parts of one (b,h) group (fwd_tail_plan: <= n_sm per launch)
constexpr uint32_t kIdxBits = 14, kIdxMask = (1u << kIdxBits) - 1u;       // rows / slots < 16384

// The key-norm pass reads every key of a (b,h) group once (N * 256 B) to save ~6% of the group's
// attention work (tiles * 8.4 MFLOP): measured on B200 that pays from about N / 8 active tiles per
// group, i.e. NKB * 16 (N = 128 NKB); sparser groups keep the exact running max instead.
__host__ __device__ __forceinline__ bool key_norm_wanted(int active_tiles, int NKB) {
  return active_tiles >= 16 * NKB;
}

// shared-memory sort of s[0, n2), n2 a power of two, DESCENDING (zeros, the padding, end up last)
__device__ void bitonic_sort_desc(uint32_t* s, int n2) {
  for (int k = 2; k <= n2; k <<= 1) {
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int i = threadIdx.x; i < n2; i += blockDim.x) {
        const int x = i ^ j;
        if (x > i) {
          const uint32_t a = s[i], b = s[x];
          const bool desc = (i & k) == 0;
          if (desc ? (a < b) : (a > b)) { s[i] = b; s[x] = a; }
        }
      }
      __syncthreads();
    }
  }
}

// Descending sort of the non-zero, pairwise distinct keys in s[0, n) (zeros = padding, last). Up to
// kRankSortMax keys: rank by counting (n broadcast reads per key, two barriers) into `alt`, and the
// two buffers swap roles; the bitonic network needs ~log^2(n)/2 barriers, which at a few hundred
// keys is most of the pre-pass. Larger problems (alt == nullptr) take the network.
constexpr int kRankSortMax = 2048;
__device__ void sort_desc(uint32_t*& s, uint32_t*& alt, int n, int n2) {
  if (alt == nullptr) {
    bitonic_sort_desc(s, n2);
    return;
  }
  for (int i = threadIdx.x; i < n2; i += blockDim.x) alt[i] = 0u;
  __syncthreads();
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    const uint32_t key = s[i];
    if (key == 0u) continue;
    int pos = 0;
    for (int j = 0; j < n; ++j) pos += s[j] > key;
    alt[pos] = key;
  }
  __syncthreads();
  uint32_t* t = s;
  s = alt;
  alt = t;
}

__device__ __forceinline__ int pow2_at_least(int n) {
  int p = 32;
  while (p < n) p <<= 1;
  return p;
}


// grid = B*H blocks. Builds the items of group (b,h), sorted by cost (active tiles) descending:
// local_items[bh][pos] = {cost, ua | ub << 16, part slot or -1, 0} (ub =
// 0xFFFF: single-row item); head_cost[bh] = active tiles of the group; head_count[bh] = its number
// of items, the last head_tail[bh] of which (the parts of the group's lightest items, plan.rem of
// them over all groups) belong at the end of the issue order; tasks[] lists the rows issued in parts.
// Dynamic shared memory: keys[n2] (uint32), then pop[NQB], ia[slots], ib[slots] (uint16).
__global__ void __launch_bounds__(kSortThreads)
schedule_items_kernel(const uint32_t* __restrict__ mask_bits, int H, int NQB, int NKB, int W,
                      int pair_rows, int split_rows, int split_leftover, int plan_rem, int plan_parts, int n2,
                      int32_t* __restrict__ head_cost, int32_t* __restrict__ head_count,
                      int32_t* __restrict__ head_tail, int4* __restrict__ local_items,
                      int4* __restrict__ tasks, uint32_t* __restrict__ part_mask,
                      float* __restrict__ kmax2) {
  extern __shared__ uint32_t s_dyn[];
  const int slots = NQB + 2;
  const bool small = n2 <= kRankSortMax;             // then a second key buffer follows the first
  uint32_t* s_keys = s_dyn;
  uint32_t* s_alt = small ? s_dyn + n2 : nullptr;
  uint16_t* s_pop = reinterpret_cast<uint16_t*>(s_dyn + (small ? 2 : 1) * n2);
  uint16_t* s_a = s_pop + ((NQB + 1) & ~1);
  uint16_t* s_b = s_a + slots;
  __shared__ int s_total, s_pool, s_count;
  const int bh = blockIdx.x, h = bh % H;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t* rows = mask_bits + static_cast<size_t>(h) * NQB * W;
  const uint32_t tail_mask = (NKB & 31) ? ((1u << (NKB & 31)) - 1u) : 0xFFFFFFFFu;
  if (threadIdx.x == 0) {
    s_total = 0;
    s_pool = 0;
    s_count = 0;
  }
  for (int i = threadIdx.x; i < n2; i += blockDim.x) s_keys[i] = 0u;
  for (int i = threadIdx.x; i < slots; i += blockDim.x) s_a[i] = s_b[i] = 0xFFFFu;
  griddep_wait();        // (launched programmatically: the mask may come from the kernel just before)
  __syncthreads();

  // ---- popcount of every row (one warp per row, lanes over the words)
  int my_total = 0;
  for (int r0 = warp; r0 < NQB; r0 += 4 * (kSortThreads / 32)) {     // four rows (loads) in flight per warp
    int c[4] = {0, 0, 0, 0};
    for (int w = lane; w < W; w += 32) {
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int r = r0 + i * (kSortThreads / 32);
        uint32_t x = r < NQB ? __ldg(rows + static_cast<size_t>(r) * W + w) : 0u;
        if (w == W - 1) x &= tail_mask;
        c[i] += __popc(x);
      }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int r = r0 + i * (kSortThreads / 32);
      const int ci = __reduce_add_sync(0xFFFFFFFFu, c[i]);
      if (lane == 0 && r < NQB) {
        s_pop[r] = static_cast<uint16_t>(ci);
        my_total += ci;
      }
    }
  }
  if (lane == 0) atomicAdd(&s_total, my_total);
  __syncthreads();

  const int n_adj = pair_rows ? NQB / 2 : 0;     // slots [0, n_adj): adjacent pairs; then pool pairs
  if (pair_rows) {
    // ---- adjacent pairs: kept when balanced (the lighter row has at least ~0.4 of the heavier
    // one's tiles: below that, running the heavy row alone for most of the item costs more than
    // the shared K/V tiles save), otherwise both rows go to the pool
    for (int i = threadIdx.x; i < n_adj; i += blockDim.x) {
      const int pa = s_pop[2 * i], pb = s_pop[2 * i + 1];
      const int lo = min(pa, pb), hi = max(pa, pb);
      if (5 * lo + 8 >= 2 * hi) {
        s_a[i] = static_cast<uint16_t>(2 * i);
        s_b[i] = static_cast<uint16_t>(2 * i + 1);
      } else {
        const int at = atomicAdd(&s_pool, 2);
        s_keys[at] = (static_cast<uint32_t>(pa) << kIdxBits) | (kIdxMask - (2 * i));
        s_keys[at + 1] = (static_cast<uint32_t>(pb) << kIdxBits) | (kIdxMask - (2 * i + 1));
      }
    }
    if (threadIdx.x == 0 && (NQB & 1)) {
      const int at = atomicAdd(&s_pool, 1);
      s_keys[at] = (static_cast<uint32_t>(s_pop[NQB - 1]) << kIdxBits) | (kIdxMask - (NQB - 1));
    }
    __syncthreads();
    const int P = s_pool;
    if (P > 0) {
      // ---- pool: popcount descending (ties: lower row first; the keys are unique, so the order
      // does not depend on the order of the atomics above)
      sort_desc(s_keys, s_alt, P, small ? n2 : pow2_at_least(P));
      // windows of four rows: of the three ways to split {0,1,2,3} into two pairs take the one
      // with the largest total overlap; a last window of 1-3 rows pairs in order
      for (int g = warp; 4 * g < P; g += kSortThreads / 32) {
        int r[4];
        for (int i = 0; i < 4; ++i)
          r[i] = 4 * g + i < P ? static_cast<int>(kIdxMask - (s_keys[4 * g + i] & kIdxMask)) : -1;
        int p0 = 1, p1 = 2, p2 = 3;              // partner of row 0; the remaining two rows
        if (r[3] >= 0) {
          const uint32_t* m0 = rows + static_cast<size_t>(r[0]) * W;
          const uint32_t* m1 = rows + static_cast<size_t>(r[1]) * W;
          const uint32_t* m2 = rows + static_cast<size_t>(r[2]) * W;
          const uint32_t* m3 = rows + static_cast<size_t>(r[3]) * W;
          // total overlap |a & b| + |c & d| of the three pairings, over the W mask words
          int s0 = 0, s1 = 0, s2 = 0;
          for (int w = lane; w < W; w += 32) {
            const uint32_t keep = (w == W - 1) ? tail_mask : 0xFFFFFFFFu;
            const uint32_t x0 = __ldg(m0 + w) & keep, x1 = __ldg(m1 + w) & keep;
            const uint32_t x2 = __ldg(m2 + w) & keep, x3 = __ldg(m3 + w) & keep;
            s0 += __popc(x0 & x1) + __popc(x2 & x3);
            s1 += __popc(x0 & x2) + __popc(x1 & x3);
            s2 += __popc(x0 & x3) + __popc(x1 & x2);
          }
          s0 = __reduce_add_sync(0xFFFFFFFFu, s0);
          s1 = __reduce_add_sync(0xFFFFFFFFu, s1);
          s2 = __reduce_add_sync(0xFFFFFFFFu, s2);
          int best = s0;
          if (s1 > best) { best = s1; p0 = 2; p1 = 1; p2 = 3; }
          if (s2 > best) { p0 = 3; p1 = 1; p2 = 2; }
        }
        if (lane == 0) {
          // a row left without a partner becomes a split item (ub = ua): its key blocks alternate
          // between the kernel's two tiles, so that both softmax warpgroups work on it (a single-row
          // item, ub = 0xFFFF, when the launch runs the lean kernel build, which has no split items)
          const int s = n_adj + 2 * g;
          s_a[s] = static_cast<uint16_t>(r[0]);
          s_b[s] = static_cast<uint16_t>(r[p0] >= 0 ? r[p0] : (split_leftover ? r[0] : 0xFFFF));
          if (r[p1] >= 0) {
            s_a[s + 1] = static_cast<uint16_t>(r[p1]);
            s_b[s + 1] = static_cast<uint16_t>(r[p2] >= 0 ? r[p2] : (split_leftover ? r[p1] : 0xFFFF));
          }
        }
      }
      __syncthreads();
      for (int i = threadIdx.x; i < n2; i += blockDim.x) s_keys[i] = 0u;
      __syncthreads();
    }
  } else {
    for (int i = threadIdx.x; i < NQB; i += blockDim.x) s_a[i] = static_cast<uint16_t>(i);
    __syncthreads();
  }

  // ---- items by cost descending (ties: lower slot first); empty slots keep key 0 and sort last
  const int used = pair_rows ? slots : NQB;       // slots that may hold an item
  int mine = 0;
  for (int s = threadIdx.x; s < min(used, slots); s += blockDim.x) {
    const int a = s_a[s], b = s_b[s];
    if (a == 0xFFFF) continue;
    const int cost = s_pop[a] + ((b != 0xFFFF && b != a) ? s_pop[b] : 0);
    s_keys[s] = (static_cast<uint32_t>(cost + 1) << kIdxBits) | (kIdxMask - s);
    ++mine;
  }
  if (mine) atomicAdd(&s_count, mine);
  __syncthreads();
  sort_desc(s_keys, s_alt, min(used, slots), n2);
  const int count = s_count;
  // HEAVY items: at least four times the group's mean item and 64 key blocks (BASELINE.json's
  // adversarial mask: the pairs of fully dense rows next to diagonal-only ones). They lead the
  // sorted list; the issue order takes the heavy items of ALL groups first, so that the launch does
  // not end on the last group's long items while the other SMs have run out of work.
  __shared__ int s_heavy;
  if (threadIdx.x == 0) s_heavy = 0;
  __syncthreads();
  {
    int mine_heavy = 0;
    for (int pos = threadIdx.x; pos < count; pos += blockDim.x) {
      const long long cost = static_cast<long long>(s_keys[pos] >> kIdxBits) - 1;
      mine_heavy += (cost >= 64 && cost * count >= 4LL * s_total) ? 1 : 0;
    }
    if (mine_heavy) atomicAdd(&s_heavy, mine_heavy);
  }
  __syncthreads();
  // this group's share of the plan's rows-in-parts: tasks [t0, t0 + n_tail) of plan_rem
  const long long BH = static_cast<long long>(gridDim.x);
  const int t0 = static_cast<int>(bh * static_cast<long long>(plan_rem) / BH);
  const int t1 = static_cast<int>((bh + 1) * static_cast<long long>(plan_rem) / BH);
  // (the group's record arrays hold NQB entries: count + n_tail * (parts - 1) must fit)
  const int n_tail = min(min(min(t1 - t0, count), kMaxTail),
                         plan_parts > 1 ? (NQB - count) / (plan_parts - 1) : 0);
  const int n_main = count - n_tail;
  for (int k = n_tail + threadIdx.x; k < t1 - t0; k += blockDim.x) tasks[t0 + k] = make_int4(-1, 0, 0, 0);
  for (int pos = threadIdx.x; pos < n_main; pos += blockDim.x) {
    const uint32_t key = s_keys[pos];
    const int s = static_cast<int>(kIdxMask - (key & kIdxMask));
    // single-row items of the tcgen05 kernel are SPLIT items (ub = ua): the row's key blocks go to
    // the kernel's two tiles in turn, so both softmax warpgroups work on the one row
    const int ub = (!pair_rows && split_rows) ? s_a[s] : s_b[s];
    local_items[static_cast<size_t>(bh) * NQB + pos] =
        make_int4(static_cast<int>(key >> kIdxBits) - 1, s_a[s] | (ub << 16), -1, 0);
  }
  // ---- the group's lightest items, in parts. One warp per item: the union of its bit-rows is cut
  // where its key blocks' running count passes c * i / parts (items of fewer than kMinPartBlocks key
  // blocks per part take fewer parts, or stay whole)
  __shared__ int s_np[kMaxTail], s_cut[kMaxTail][3], s_at[kMaxTail + 1];
  for (int k = warp; k < n_tail; k += kSortThreads / 32) {
    const int s = static_cast<int>(kIdxMask - (s_keys[n_main + k] & kIdxMask));
    const int a = s_a[s], b = s_b[s];
    const uint32_t* ma = rows + static_cast<size_t>(a) * W;
    const uint32_t* mb = (b != 0xFFFF && b != a) ? rows + static_cast<size_t>(b) * W : ma;
    int c = 0;
    for (int w = lane; w < W; w += 32) {
      const uint32_t keep = (w == W - 1) ? tail_mask : 0xFFFFFFFFu;
      c += __popc((__ldg(ma + w) | __ldg(mb + w)) & keep);
    }
    c = __reduce_add_sync(0xFFFFFFFFu, c);
    int np = plan_parts;
    while (np > 1 && c < kMinPartBlocks * np) np >>= 1;
    // key block holding the union's bit of rank r_i = c * i / np: part i starts there
    int done = 0, next = 1;
    for (int w0 = 0; w0 < W && next < np; w0 += 32) {
      const int w = w0 + lane;
      uint32_t x = 0u;
      if (w < W) x = (__ldg(ma + w) | __ldg(mb + w)) & ((w == W - 1) ? tail_mask : 0xFFFFFFFFu);
      const int n = __popc(x);
      int incl = n;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += v;
      }
      const int chunk = __shfl_sync(0xFFFFFFFFu, incl, 31);
      while (next < np) {
        const int r = static_cast<int>(static_cast<long long>(c) * next / np) - done;   // rank inside this chunk
        if (r >= chunk) break;
        const bool mine = r >= incl - n && r < incl;
        const uint32_t who = __ballot_sync(0xFFFFFFFFu, mine);
        const int bit = mine ? static_cast<int>(__fns(x, 0, r - (incl - n) + 1)) : 0;
        const int kb = __shfl_sync(0xFFFFFFFFu, w * 32 + bit, __ffs(who) - 1);
        if (lane == 0) s_cut[k][next - 1] = kb;
        ++next;
      }
      done += chunk;
    }
    // too short for parts, but a real pair: its two rows become two SINGLE-ROW items (ub = 0xFFFF, the
    // kernel's second tile idle) at the end of the order -- about 0.6 of the pair's time each, which
    // is what the partly filled last round then takes (np = -2 marks it)
    if (np == 1 && b != 0xFFFF && b != a && min(s_pop[a], s_pop[b]) >= kMinSingleBlocks) np = -2;
    if (lane == 0) s_np[k] = np;
  }
  __syncthreads();
  // items that stay whole keep their place in the group's list (their K/V is in L2 while the group
  // runs); only real parts move to the end of the issue order
  __shared__ int s_main_end;
  if (threadIdx.x == 0) {
    int at = n_main;
    for (int k = 0; k < n_tail; ++k)
      if (s_np[k] == 1) s_at[k] = at++;
    s_main_end = at;
    for (int k = 0; k < n_tail; ++k)
      if (s_np[k] != 1) {
        s_at[k] = at;
        at += abs(s_np[k]);
      }
    s_at[n_tail] = at;
  }
  __syncthreads();
  for (int k = warp; k < n_tail; k += kSortThreads / 32) {
    const uint32_t key = s_keys[n_main + k];
    const int s = static_cast<int>(kIdxMask - (key & kIdxMask));
    const int rows_ab = s_a[s] | (s_b[s] << 16);
    const int np = s_np[k], slot0 = (t0 + k) * plan_parts;
    if (np == -2) {
      if (lane < 2) {
        const int u = lane == 0 ? (rows_ab & 0xFFFF) : ((rows_ab >> 16) & 0xFFFF);
        local_items[static_cast<size_t>(bh) * NQB + s_at[k] + lane] =
            make_int4(s_pop[u], u | (0xFFFF << 16), -1, 0);
      }
      if (lane == 0) tasks[t0 + k] = make_int4(-1, rows_ab, 1, slot0);
      continue;
    }
    if (lane < np)
      local_items[static_cast<size_t>(bh) * NQB + s_at[k] + lane] =
          make_int4(static_cast<int>(key >> kIdxBits) - 1, rows_ab, np > 1 ? slot0 + lane : -1, 0);
    if (np > 1) {
      // the parts' bit-rows: rows a and b with the bits of part i's key range [lo_i, hi_i) only
      const int a = rows_ab & 0xFFFF, b = (rows_ab >> 16) & 0xFFFF;
      const uint32_t* ma = rows + static_cast<size_t>(a) * W;
      const uint32_t* mb = rows + static_cast<size_t>(b != 0xFFFF ? b : a) * W;
      for (int i = 0; i < np; ++i) {
        const int lo = i == 0 ? 0 : s_cut[k][i - 1];
        const int hi = i == np - 1 ? 32 * W : s_cut[k][i];
        uint32_t* dst = part_mask + static_cast<size_t>(2 * (slot0 + i)) * W;
        for (int w = lane; w < W; w += 32) {
          const int l = max(lo - 32 * w, 0), h2 = min(hi - 32 * w, 32);
          const uint32_t m = l < h2 ? (0xFFFFFFFFu << l) & (0xFFFFFFFFu >> (32 - h2)) : 0u;
          dst[w] = __ldg(ma + w) & m;
          dst[W + w] = __ldg(mb + w) & m;
        }
      }
    }
    if (lane == 0) tasks[t0 + k] = make_int4(np > 1 ? bh : -1, rows_ab, np, slot0);
  }
  if (threadIdx.x == 0) {
    const int at = s_at[n_tail];
    head_cost[bh] = s_total;
    head_count[bh] = at;
    head_tail[bh] = (at - s_main_end) | (min(s_heavy, n_main) << 16);
    // the key-norm pass (next on the stream) takes the max into kmax2[bh] -- or skips the group and
    // leaves the "no bound" mark when it is too sparse for the pass to pay (key_norm_wanted)
    kmax2[bh] = key_norm_wanted(s_total, NKB) ? 0.f : -1.f;
  }
}

// kmax2[bh] = max over the valid keys j of |k_j|^2 (D = 128), rows [r0, r1). Half a warp per key row:
// 16 lanes x 16 bytes = one 256 B row per load, fully coalesced; 4 shuffles fold the 16 partial sums.
// The forward kernel turns it into the Cauchy-Schwarz bound scale * |q_i| * max_j |k_j| >= every
// score of query row i, which lets it fix the softmax reference point of a row for a whole item.
constexpr int kFlatThreads = 256;
constexpr int kNormRowsPerBlock = 256;
__device__ __forceinline__ void key_norm_slice(const __nv_bfloat16* __restrict__ k, int N, int r0, int r1,
                                               int bh, float* __restrict__ kmax2) {
  const int half = threadIdx.x >> 4, sub = threadIdx.x & 15;       // 16 half-warps per block
  const uint4* base = reinterpret_cast<const uint4*>(k + static_cast<size_t>(bh) * N * 128);
  float best = 0.f;
#pragma unroll 4
  for (int rb = r0; rb < r1; rb += kFlatThreads / 16) {       // uniform trip count (shuffles inside)
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

// grid = (X, B*H). Block (x, bh): (1) if `flatten`, copies items [256 x, 256 x + 256) of group bh to
// their place in the issue order -- the groups go heaviest first (ties: lower id), so the group's
// first item sits at the sum of the item counts of the groups ahead of it, which every copying block
// works out for itself in O(B*H / 256) steps; block (0,0) also zeroes the cursor and publishes the
// total item count; (2) if `k` is given, takes key rows [1024 x, 1024 x + 1024) of the group into
// kmax2[bh] (one launch instead of two: the forward call is launch-latency bound on short sequences).
__global__ void __launch_bounds__(kFlatThreads)
schedule_flatten_kernel(const int32_t* __restrict__ head_cost, const int32_t* __restrict__ head_count,
                        const int32_t* __restrict__ head_tail, const int4* __restrict__ local_items,
                        int BH, int NQB, int flatten,
                        int4* __restrict__ items, int32_t* __restrict__ cursor,
                        int32_t* __restrict__ n_items, const __nv_bfloat16* __restrict__ k, int N,
                        int n_valid, float* __restrict__ kmax2) {
  const int bh = blockIdx.y;
  griddep_wait();
  if (flatten) {
    const int count = __ldg(head_count + bh);
    const bool first = blockIdx.x == 0 && bh == 0;
    if (static_cast<int>(blockIdx.x) * kFlatThreads < count || first) {
      // the order: every group's HEAVY items (head_tail >> 16 of them, the first of its list), then
      // every group's other whole items, then the groups' parts (head_tail & 0xFFFF, the last of its list)
      __shared__ int s_sum[6];        // items / heavy / tail: of the groups ahead, of all groups
      if (threadIdx.x < 6) s_sum[threadIdx.x] = 0;
      __syncthreads();
      const int cg = __ldg(head_cost + bh);
      int v[6] = {0, 0, 0, 0, 0, 0};
      for (int j = threadIdx.x; j < BH; j += kFlatThreads) {
        const int cj = __ldg(head_cost + j), nj = __ldg(head_count + j), pj = __ldg(head_tail + j);
        const int hj = pj >> 16, tj = pj & 0xFFFF;
        v[3] += nj;
        v[4] += hj;
        v[5] += tj;
        if (cj > cg || (cj == cg && j < bh)) {
          v[0] += nj;
          v[1] += hj;
          v[2] += tj;
        }
      }
#pragma unroll
      for (int i = 0; i < 6; ++i) {
        v[i] = __reduce_add_sync(0xFFFFFFFFu, v[i]);
        if ((threadIdx.x & 31) == 0 && v[i]) atomicAdd(&s_sum[i], v[i]);
      }
      __syncthreads();
      const int pos = blockIdx.x * kFlatThreads + threadIdx.x;
      if (pos < count) {
        const int4 rec = __ldg(local_items + static_cast<size_t>(bh) * NQB + pos);
        const int packed = __ldg(head_tail + bh);
        const int n_heavy = packed >> 16, n_main = count - (packed & 0xFFFF);
        const int all = s_sum[3], all_heavy = s_sum[4], all_tail = s_sum[5];
        int at;
        if (pos < n_heavy) at = s_sum[1] + pos;
        else if (pos < n_main) at = all_heavy + (s_sum[0] - s_sum[1] - s_sum[2]) + (pos - n_heavy);
        else at = (all - all_tail) + s_sum[2] + (pos - n_main);
        items[at] = make_int4(bh, rec.y, rec.z, 0);
      }
      const int s_all = s_sum[3];
      if (first && threadIdx.x == 0) {
        cursor[0] = 0;
        cursor[2] = cursor[3] = 0;    // softmax-path counters of the coming call
        *n_items = s_all;
      }
    }
  }
  if (k != nullptr) {
    const int r0 = blockIdx.x * kNormRowsPerBlock;
    const int r1 = min(r0 + kNormRowsPerBlock, n_valid);
    if (!key_norm_wanted(__ldg(head_cost + bh), N / 128)) {
      if (blockIdx.x == 0 && threadIdx.x == 0) kmax2[bh] = -1.f;   // (the reuse form zero-fills kmax2 first)
    } else if (r0 < r1) {
      key_norm_slice(k, N, r0, r1, bh, kmax2);
    }
  }
}

// grid = (plan.rem, 2), 256 threads: block (t, tile) merges the parts of query block ua (tile 0) / ub
// (tile 1) of task t. A part holds the softmax over its key range: normalised O_i (bf16) and lse_i;
// over the whole row  lse = m + ln sum_i e^(lse_i - m),  O = sum_i e^(lse_i - lse) O_i, summed in part
// order. A warp takes 16 rows, row by row across the 256 bytes of a row (8 bytes per lane), four rows'
// loads in flight; lane r holds the weights of the warp's row r. Launched with programmatic stream
// serialization: the launch overlaps the attention kernel, griddepcontrol.wait orders the reads.
__global__ void __launch_bounds__(256)
combine_parts_kernel(const int4* __restrict__ tasks, const __nv_bfloat16* __restrict__ part_out,
                     const float* __restrict__ part_lse, int N, __nv_bfloat16* __restrict__ out,
                     float* __restrict__ lse) {
  griddep_wait();
  const int4 task = __ldg(tasks + blockIdx.x);              // {b*H + h, ua | ub << 16, parts, first slot}
  const int tile = blockIdx.y;
  const int ua = task.y & 0xFFFF, ub = (task.y >> 16) & 0xFFFF;
  if (task.x < 0 || (tile == 1 && (ub == 0xFFFF || ub == ua))) return;   // whole item / one row only
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int np = task.z;
  const int row = warp * 16 + (lane & 15);                  // lanes 16-31 mirror 0-15
  float l[4], m = -INFINITY;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    l[i] = i < np ? __ldcg(part_lse + (static_cast<size_t>(2 * (task.w + i) + tile) * 128 + row)) : -INFINITY;
    m = fmaxf(m, l[i]);
  }
  float wgt[4], sum = 0.f;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    wgt[i] = l[i] > -INFINITY ? expf(l[i] - m) : 0.f;
    sum += wgt[i];
  }
  const float inv = sum > 0.f ? 1.f / sum : 0.f;
#pragma unroll
  for (int i = 0; i < 4; ++i) wgt[i] *= inv;
  const size_t grow0 = static_cast<size_t>(task.x) * N + static_cast<size_t>(tile == 0 ? ua : ub) * 128 + warp * 16;
  if (lane < 16) lse[grow0 + lane] = sum > 0.f ? m + logf(sum) : -INFINITY;
#pragma unroll 1
  for (int r0 = 0; r0 < 16; r0 += 4) {
    uint2 x[4][4];
#pragma unroll
    for (int rr = 0; rr < 4; ++rr)
#pragma unroll
      for (int i = 0; i < 4; ++i)
        if (i < np)
          x[rr][i] = __ldcg(reinterpret_cast<const uint2*>(
                                part_out + (static_cast<size_t>(2 * (task.w + i) + tile) * 128 + warp * 16 + r0 + rr) * 128) +
                            lane);
#pragma unroll
    for (int rr = 0; rr < 4; ++rr) {
      float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float sc = __shfl_sync(0xFFFFFFFFu, wgt[i], r0 + rr);
        if (i < np) {
          acc[0] = fmaf(__uint_as_float(x[rr][i].x << 16), sc, acc[0]);
          acc[1] = fmaf(__uint_as_float(x[rr][i].x & 0xFFFF0000u), sc, acc[1]);
          acc[2] = fmaf(__uint_as_float(x[rr][i].y << 16), sc, acc[2]);
          acc[3] = fmaf(__uint_as_float(x[rr][i].y & 0xFFFF0000u), sc, acc[3]);
        }
      }
      const __nv_bfloat162 lo = __floats2bfloat162_rn(acc[0], acc[1]), hi = __floats2bfloat162_rn(acc[2], acc[3]);
      reinterpret_cast<uint2*>(out + (grow0 + r0 + rr) * 128)[lane] =
          make_uint2(*reinterpret_cast<const uint32_t*>(&lo), *reinterpret_cast<const uint32_t*>(&hi));
    }
  }
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

cudaError_t launch_schedule(const FwdParams& p, const FwdWorkspace& w, int rpi, TailPlan plan,
                            cudaStream_t st, int* n_launch, bool reuse) {
  const int BH = p.B * p.H;
  const bool norms = p.D == 128 && p.kmax2 != nullptr;   // the tcgen05 kernel's score bound needs max |k|^2
  cudaError_t e;
  if (reuse) {
    // the work list in the workspace is still valid (same mask): only reset what a call consumes
    e = cudaMemsetAsync(w.cursor, 0, sizeof(int32_t), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(w.stats, 0, 2 * sizeof(int32_t), st);
    if (e == cudaSuccess && norms) e = cudaMemsetAsync(w.kmax2, 0, static_cast<size_t>(BH) * sizeof(float), st);
    if (e != cudaSuccess) return e;
  } else {
    int n2 = 32;
    while (n2 < p.NQB + 2) n2 <<= 1;
    const size_t smem = static_cast<size_t>(n2) * 4 * (n2 <= kRankSortMax ? 2 : 1) +
                        (static_cast<size_t>((p.NQB + 1) & ~1) + 2 * (p.NQB + 2)) * 2;
    if (smem > 48 * 1024) {
      e = ensure_dynamic_smem(kSmemScheduleItems, reinterpret_cast<const void*>(schedule_items_kernel),
                              200 * 1024);
      if (e != cudaSuccess) return e;
    }
    e = launch_pdl(schedule_items_kernel, dim3(BH), dim3(kSortThreads), smem, st, p.mask_bits, p.H, p.NQB, p.NKB,
                   p.W, rpi == 2 ? 1 : 0, p.split_rows, p.lean_items ? 0 : 1, rpi == 2 ? plan.rem : 0, plan.parts, n2,
                   w.head_cost,
                   w.head_count, w.head_tail, w.local_items, w.tasks, w.part_mask, w.kmax2);
    if (e != cudaSuccess) return e;
    *n_launch += 1;
  }
  if (!reuse || norms) {
    const int xf = reuse ? 0 : (p.NQB + kFlatThreads - 1) / kFlatThreads;
    const int xn = norms ? (p.n_valid + kNormRowsPerBlock - 1) / kNormRowsPerBlock : 0;
    const dim3 grid(xf > xn ? xf : xn, BH);
    const int32_t* hc = w.head_cost;
    const int32_t* hn = w.head_count;
    const int32_t* ht = w.head_tail;
    const int4* li = w.local_items;
    e = launch_pdl(schedule_flatten_kernel, grid, dim3(kFlatThreads), 0, st, hc, hn, ht, li, BH, p.NQB,
                   reuse ? 0 : 1, w.items, w.cursor, w.n_items, norms ? p.k : nullptr, p.N, p.n_valid, w.kmax2);
    if (e != cudaSuccess) return e;
    *n_launch += 1;
  }
  return cudaGetLastError();
}

cudaError_t launch_combine_parts(const FwdParams& p, const FwdWorkspace& w, TailPlan plan,
                                 cudaStream_t st, int* n_launch) {
  if (plan.rem <= 0) return cudaSuccess;
  const int4* tasks = w.tasks;
  const __nv_bfloat16* po = w.part_out;
  const float* pl = w.part_lse;
  cudaError_t e = launch_pdl(combine_parts_kernel, dim3(plan.rem, 2), dim3(256), 0, st, tasks, po, pl, p.N, p.out,
                             p.lse);
  if (e != cudaSuccess) return e;
  *n_launch += 1;
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

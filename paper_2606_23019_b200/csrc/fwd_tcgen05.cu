// fwd_tcgen05.cu -- block-sparse attention forward for (D,Bq,Bk) = (128,128,128) on sm_100a:
// TMA-fed shared-memory ring, tcgen05.mma with accumulators in TMEM, warp-specialised online softmax.
//
// What it computes: the crm kernel of the paper (Sec. 4.3.2) -- FlashAttention's
// forward pass with the dense KV-block iterator replaced by the CRM bit-row iterator (Alg. 2,
// PAPER.md:484-539). Masked key blocks are never loaded and never multiplied.
//
// How (this design is for B200, not the paper's):
//   * persistent grid, one CTA per SM; a work item is a PAIR of query blocks (ua, ub) of one
//     (batch, head), chosen by the schedule pre-pass (adjacent blocks when their popcounts are
//     balanced, else partners of similar popcount and large bit-row overlap; schedule.cu). Items
//     are pulled from the popcount-ordered list of the pre-pass with an atomic cursor, so uneven
//     rows and heads balance out. The producer claims
//     one item ahead (2-slot scheduler ring) so the atomic's round trip hides under the current
//     item's loads; after a long item the claim is taken late instead, so that the tail of the
//     grid still goes to whichever CTA is free first.
//   * the two query tiles have different bit-rows; the CTA walks the UNION of the two rows, stages
//     each K/V tile of the union ONCE (TMA, 128B swizzle, 5-slot ring of 32 KB tiles), and issues
//     the MMAs of a tile only where that tile's own bit is set, so a key block both rows have is
//     read from L2 once.
//   * warp 0: scheduler + TMA producer; warp 1: tcgen05.mma issuer; both run converged and issue
//     through elect.sync (uniform-register UTCHMMA / UTMALDG); warp 2: TMEM allocator; warps 4-7 /
//     8-11: softmax warpgroups of query tile 0 / 1 (one thread per row).
//   * TMEM (512 columns): two S/P buffers [0,128) [128,256), O0 [256,384) O1 [384,512), fp32. P
//     (bf16, two per column) overwrites the first 64 columns of its S and feeds the PV MMA as the
//     TMEM A operand, so P never touches shared memory.
//   * (tile, key block) units are numbered in walk order; unit w uses buffer w & 1 and the issue
//     order is PV(w-2), S(w): the softmax of one unit overlaps the MMAs of its neighbours whether
//     the neighbours belong to the other tile or to the same one.
//   * softmax in the log2 domain, scale folded into one FFMA2. A row's reference point is normally
//     the Cauchy-Schwarz bound scale*|q_i|*max|k| (>= every score), fixed for the whole item: no
//     running max, no rescale. If the first key block shows the bound is too loose, the warp keeps
//     the exact running max, raised only when it grows by more than 8 (factor 256), which keeps the
//     O rescale (a TMEM round trip) off the common path; out and lse use the same reference point
//     consistently, so the result is the same softmax either way.
#include <cuda.h>

#include "common.cuh"
#include "ptx.cuh"
#include "trace.cuh"

namespace sa {
namespace {

using namespace ptx;

constexpr int kBlk = 128;                 // Bq = Bk
constexpr int kD = 128;
constexpr int kThreads = 384;
constexpr uint32_t kTileBytes = kBlk * kD * 2;      // 32 KB
constexpr uint32_t kHalfBytes = kTileBytes / 2;     // one [128][64] swizzle-128B box
#ifndef SA_SLOTS
#define SA_SLOTS 5
#endif
constexpr int kSlots = SA_SLOTS;          // K/V ring
constexpr int kSched = 2;                 // scheduler ring
constexpr int kClaimAheadUnits = 512;     // items up to this many (tile, key block) units claim their successor early
constexpr uint32_t kTmemCols = 512;
constexpr float kRescaleThreshold = 8.0f; // log2 units
constexpr float kBoundSlack = 64.0f;      // log2 units: how far the Cauchy-Schwarz bound may lie above
                                          // the first block's row maximum and still be used (2^-64 of
                                          // headroom is left before fp32 / bf16 flush to zero at 2^-126)
// Tunable of the softmax (default chosen by measurement on B200):
//  SA_POLY_PAIRS: of every 4 consecutive column pairs, how many take exp2 on the FMA pipe
//  (Cody-Waite split + degree-3 polynomial) instead of MUFU.EX2 -- the MUFU pipe (16/clk/SM)
//  would otherwise need as many cycles per tile as the two MMAs. Off: under the power cap the
//  extra instructions cost more than the shorter exponential phase gains.
#ifndef SA_POLY_PAIRS
#define SA_POLY_PAIRS 0
#endif
constexpr int kPolyPairs = SA_POLY_PAIRS;
static_assert(kPolyPairs >= 0 && kPolyPairs <= 4, "SA_POLY_PAIRS in 0..4");
// P is handed to the PV MMA in two pieces of 64 keys (p_full[..][0], [1]): the MMAs of the first
// keys start while the exponentials of the later ones are still being computed.
constexpr int kPChunks = 2;

// shared memory map (offsets from a 1024 B aligned base)
constexpr uint32_t kOffQ = 0;                                   // 2 query tiles
constexpr uint32_t kOffRing = 2 * kTileBytes;                   // kSlots tiles
constexpr uint32_t kOffCtl = kOffRing + kSlots * kTileBytes;    // barriers etc.
struct __align__(8) Ctl {
  uint64_t q_full, q_empty;
  uint64_t kv_full[kSlots], kv_empty[kSlots];
  uint64_t s_full[2][2], p_full[2][2][4], pv_done[2][2];   // [tile][tile-local unit & 1]
  uint64_t o_full[2], o_free[2];
  uint64_t xchg_full, xchg_empty;     // split items: warpgroup 1 has published its half / warpgroup 0 has read it
  uint64_t sched_full[kSched], sched_empty[kSched];
  int4 sched_item[kSched];            // item record (x = -1: no more work)
  uint32_t tmem_base;
};
constexpr uint32_t kSmemBytes = kOffCtl + sizeof(Ctl) + 1024;   // + alignment slack
static_assert(kSmemBytes <= 232448, "exceeds 227 KB of dynamic shared memory");

// tcgen05 shared-memory matrix descriptors (sm_100 format: start>>4 [0,14), LBO>>4 [16,30),
// SBO>>4 [32,46), version=1 [46,48), layout type [61,64) with 2 = 128B swizzle).
//  K-major operand (Q, K: rows x 64 bf16 per box, 8-row groups 1024 B apart)
constexpr uint64_t kDescKMajor = (uint64_t(1) << 16) | (uint64_t(1024 >> 4) << 32) |
                                 (uint64_t(1) << 46) | (uint64_t(2) << 61);
//  MN-major operand (V as B of P.V: 64 head-dim columns contiguous, key rows 128 B apart,
//  8-key groups 1024 B apart (SBO), the next 64 head-dim columns one box = 16 KB further (LBO))
constexpr uint64_t kDescMNMajor = (uint64_t(kHalfBytes >> 4) << 16) | (uint64_t(1024 >> 4) << 32) |
                                  (uint64_t(1) << 46) | (uint64_t(2) << 61);
__device__ __forceinline__ uint64_t make_desc(uint64_t base, uint32_t smem_addr) {
  return base | static_cast<uint64_t>((smem_addr & 0x3FFFFu) >> 4);
}
// instruction descriptor: fp32 accumulate [4,6)=1, A,B bf16 [7,10)=[10,13)=1, B major bit 16,
// N>>3 at [17,23), M>>4 at [24,29)
constexpr uint32_t kIdescQK = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 3) << 17) |
                              ((128u >> 4) << 24);
constexpr uint32_t kIdescPV = kIdescQK | (1u << 16);

// A work item: query blocks ua (tile 0) and ub (tile 1) of one (batch, head); the schedule pre-pass
// chooses the pairs (schedule.cu). Single-row items leave tile 1 empty.
// (kFull = false: the LEAN build of the kernel, for launches whose work list holds neither split items nor
// parts -- large problems: the code of both is compiled out, which is worth ~1.5% at C4.)
template <bool kFull>
struct ItemT {
  int bh, h, ua, ub;
  bool has1;
  int row0;            // first token row of the (b,h) slab in the [B*H*N][D] view
  int part;            // >= 0: a PART of its rows (a key range of them): the bit-rows restricted to the range
                       // are rows 2 part, 2 part + 1 of p.part_mask, the results go to scratch slot `part`
  // ub == ua: a SPLIT item -- ONE query block whose key blocks are dealt to the two tiles in turn (even
  // key blocks -> tile 0, odd -> tile 1), the halves merged in the epilogue. (Derived on demand: the
  // softmax loop has no register to spare for another live flag.)
  __device__ __forceinline__ bool split() const { return kFull && ub == ua; }
};
// item record: x = b*H + h (-1: no more work), y = ua | ub << 16 (ub = 0xFFFF: no second row),
// z = scratch slot of a part (-1: the item covers its rows' whole bit-rows and writes out / lse itself)
template <bool kFull>
__device__ __forceinline__ ItemT<kFull> decode_item(const FwdParams& p, int4 rec) {
  ItemT<kFull> it;
  it.bh = rec.x;
  it.h = it.bh % p.H;
  it.ua = rec.y & 0xFFFF;
  it.ub = (rec.y >> 16) & 0xFFFF;
  it.has1 = it.ub != 0xFFFF;
  it.row0 = it.bh * p.N;
  it.part = kFull ? rec.z : -1;
  return it;
}

// Debug log of the walk (sa_debug_fwd_walk; p.walk_log is null in every other call and the product
// kernel is compiled without these stores). int32 regions, rows indexed by b*H*NQB + h*NQB + u:
//   wg_cnt[rows], wg_info[rows] = (partner + 1) << 1 | tile, wg_seq[rows][NKB] = unit << 16 | key block
//   (what the softmax warpgroup of the row's tile consumed, unit = number in the item's walk order),
//   is_cnt[rows], is_seq[rows][2*NKB] = tile << 15 | key block (what the MMA issuer issued for the
//   item whose tile 0 is this row, in issue order).
struct WalkLog {
  int32_t* base;
  size_t rows, nkb;
  __device__ explicit WalkLog(const FwdParams& p)
      : base(p.walk_log), rows(static_cast<size_t>(p.B) * p.H * p.NQB), nkb(p.NKB) {}
  __device__ int32_t* wg_cnt() const { return base; }
  __device__ int32_t* wg_info() const { return base + rows; }
  __device__ int32_t* wg_seq(size_t row) const { return base + 2 * rows + row * nkb; }
  __device__ int32_t* is_cnt() const { return base + 2 * rows + rows * nkb; }
  __device__ int32_t* is_seq(size_t row) const { return base + 3 * rows + rows * nkb + row * 2 * nkb; }
};

// word w of the bit-row of query block u (0 beyond the grid), stray high bits cleared; for a part,
// of the row's copy that holds the part's key range only (written by the schedule pre-pass)
__device__ __forceinline__ uint32_t row_word(const FwdParams& p, int h, int u, int w, bool exists,
                                             int part, int tile) {
  if (!exists) return 0u;
  const uint32_t* row = part < 0 ? p.mask_bits + (static_cast<size_t>(h) * p.NQB + u) * p.W
                                 : p.part_mask + static_cast<size_t>(2 * part + tile) * p.W;
  uint32_t x = __ldg(row + w);
  if (w == p.W - 1 && (p.NKB & 31)) x &= (1u << (p.NKB & 31)) - 1u;
  return x;
}

// The two bit-rows of a work item, held by the warp: lane l keeps words (base + l) and (base + 32 + l)
// of each row, fetched with one coalesced load per 64 words; word w is then a shuffle away instead of
// a dependent global load per word (at low density most words hold 0-2 key blocks, and a load per
// word put an L2 round trip into every role's walk). The shuffle's source lane is warp-uniform, so
// the result is too.
struct RowWalk {
  uint32_t a0 = 0, a1 = 0, b0 = 0, b1 = 0;
  template <class Item>
  __device__ __forceinline__ void load(const FwdParams& p, const Item& it, int base, int lane) {
    const int w0 = base + lane, w1 = base + 32 + lane;
    a0 = w0 < p.W ? row_word(p, it.h, it.ua, w0, true, it.part, 0) : 0u;
    a1 = w1 < p.W ? row_word(p, it.h, it.ua, w1, true, it.part, 0) : 0u;
    if (it.split()) {                    // one row, its key blocks alternating between the tiles
      b0 = a0 & 0xAAAAAAAAu;
      b1 = a1 & 0xAAAAAAAAu;
      a0 &= 0x55555555u;
      a1 &= 0x55555555u;
    } else {
      b0 = w0 < p.W ? row_word(p, it.h, it.ub, w0, it.has1, it.part, 1) : 0u;
      b1 = w1 < p.W ? row_word(p, it.h, it.ub, w1, it.has1, it.part, 1) : 0u;
    }
  }
  // number of set bits of each row within the loaded 64 words
  __device__ __forceinline__ void counts(uint32_t& n0, uint32_t& n1) const {
    n0 = __reduce_add_sync(0xFFFFFFFFu, __popc(a0) + __popc(a1));
    n1 = __reduce_add_sync(0xFFFFFFFFu, __popc(b0) + __popc(b1));
  }
  __device__ __forceinline__ uint32_t row0(int w) const {
    return __shfl_sync(0xFFFFFFFFu, (w & 32) ? a1 : a0, w & 31);
  }
  __device__ __forceinline__ uint32_t row1(int w) const {
    return __shfl_sync(0xFFFFFFFFu, (w & 32) ? b1 : b0, w & 31);
  }
};

struct Ring {
  int slot = 0;
  uint32_t phase = 0;
  __device__ __forceinline__ void advance() {
    if (++slot == kSlots) { slot = 0; phase ^= 1u; }
  }
};

// ------------------------------------------------------------------ warp 0: scheduler + TMA
// Runs on every lane of warp 0 (converged); elect.sync inside the _e wrappers picks the issuer.
template <bool kFull>
__device__ void producer(const FwdParams& p, Ctl* ctl, uint32_t smem_base, const CUtensorMap* tm_q,
                         const CUtensorMap* tm_k, const CUtensorMap* tm_v, int lane) {
  Ring ring;
  uint32_t q_phase = 0;
  int sched_n = 0;
  // Work items are claimed ONE AHEAD: while the loads of item n are issued, item n+1 has already
  // been taken from the list and published in the 2-slot scheduler ring, so that at the end of an
  // item nobody waits for the atomic and the list lookup (two dependent global round trips, ~3 us
  // of idle tensor pipe per item otherwise). The list is longest-first inside a head, so the items
  // claimed early near the end are the light ones and the tail stays short.
  const int n_items = __ldg(p.n_items_dev);
  auto claim_and_publish = [&]() {
    int idx = 0;
    if (lane == 0) idx = atomicAdd(p.counter, 1);
    idx = __shfl_sync(0xFFFFFFFFu, idx, 0);
    const int4 it_id = idx < n_items ? __ldg(p.items + idx) : make_int4(-1, 0, -1, 0);
    const int ss = sched_n % kSched;
    mbar_wait(smem_u32(&ctl->sched_empty[ss]), ((sched_n / kSched) & 1) ^ 1u, 1);
    if (lane == 0) {
      ctl->sched_item[ss] = it_id;
      mbar_arrive(smem_u32(&ctl->sched_full[ss]));
    }
    __syncwarp();
    ++sched_n;
    return it_id;
  };
  int4 next_item = claim_and_publish();
  for (;;) {
    const int4 item = next_item;
    if (item.x < 0) break;
    const ItemT<kFull> it = decode_item<kFull>(p, item);
    // ... unless this item is a long one (a held-back item would then wait that long while another
    // CTA may be idle): long items claim their successor only when their own loads are out
    RowWalk rw;
    uint32_t units = 0;
    for (int base = 0; base < p.W; base += 64) {
      uint32_t n0, n1;
      rw.load(p, it, base, lane);
      rw.counts(n0, n1);
      units += n0 + n1;
    }
    const bool ahead = units <= static_cast<uint32_t>(kClaimAheadUnits);
    if (ahead) next_item = claim_and_publish();

    mbar_wait(smem_u32(&ctl->q_empty), q_phase ^ 1u, 2);
    const uint32_t qf = smem_u32(&ctl->q_full);
    const int q_tiles = (it.has1 && !it.split()) ? 2 : 1;      // a split item has one query tile
    mbar_expect_tx_e(qf, q_tiles * kTileBytes);
    for (int t = 0; t < q_tiles; ++t) {
      const uint32_t dst = smem_base + kOffQ + t * kTileBytes;
      const int y = it.row0 + (t == 0 ? it.ua : it.ub) * kBlk;
      tma_load_2d_e(dst, tm_q, 0, y, qf);
      tma_load_2d_e(dst + kHalfBytes, tm_q, 64, y, qf);
    }
    q_phase ^= 1u;

    for (int w = 0; w < p.W; ++w) {
      if ((w & 63) == 0 && (w > 0 || p.W > 64)) rw.load(p, it, w, lane);
      uint32_t x = rw.row0(w) | rw.row1(w);
      while (x) {
        const int j = w * 32 + (__ffs(x) - 1);
        x &= x - 1u;
        const int y = it.row0 + j * kBlk;
#pragma unroll
        for (int kv = 0; kv < 2; ++kv) {
          const uint32_t full = smem_u32(&ctl->kv_full[ring.slot]);
          mbar_wait(smem_u32(&ctl->kv_empty[ring.slot]), ring.phase ^ 1u, 3);
          mbar_expect_tx_e(full, kTileBytes);
          const uint32_t dst = smem_base + kOffRing + ring.slot * kTileBytes;
          const CUtensorMap* tm = kv == 0 ? tm_k : tm_v;
          tma_load_2d_e(dst, tm, 0, y, full);
          tma_load_2d_e(dst + kHalfBytes, tm, 64, y, full);
          ring.advance();
        }
      }
    }
    if (!ahead) next_item = claim_and_publish();
  }
  // every MMA that reads shared memory has retired before the CTA exits
  mbar_wait(smem_u32(&ctl->q_empty), q_phase ^ 1u, 4);
}

// ------------------------------------------------------------------ warp 1: MMA issuer
// One (query tile, key block) unit whose S has been issued and whose PV is still to come. Every
// address and descriptor is worked out when the unit is created, BEFORE the issuer blocks on the
// older unit's P: once P is there, nothing but waits, MMAs and commits lies between it and the
// next S (the MMA issuer is a serial resource inside the cycle S -> softmax -> PV -> next S).
struct Pend {
  uint32_t tmem_o, tmem_p;     // O_t and the unit's P (first columns of its S/P buffer)
  uint64_t vdesc;              // V tile as the MN-major B operand
  uint32_t acc;                // accumulate into O_t (0 for the tile's first unit of the item)
  uint32_t p_full, par;        // p_full[t][sel][0] (piece c at + 8 c) and its phase parity
  uint32_t pv_done;            // barrier committed after the PV
  uint32_t v_full, vphase;     // ring slot holding V: kv_full and its parity
  uint32_t o_free, ofree_par;  // first unit of a tile only (else 0): wait before overwriting O_t
  uint32_t v_empty;            // last user of the V slot (else 0): release it after the PV
  uint32_t o_full;             // last unit of the tile in its item (else 0): commit after the PV
};

// Runs on every lane of warp 1 (converged); elect.sync inside the _e wrappers picks the issuer.
//
// Units (tile t, key block j) are numbered 0,1,2,... in walk order (ascending j over the union of
// the two bit-rows, tile 0 before tile 1), across items. Unit w computes S into buffer w & 1 -- the
// buffers alternate per UNIT, not per tile, so a run of key blocks that only one of the two query
// tiles has still ping-pongs between the two S buffers. Issue order: PV(w-2), S(w): the softmax of
// unit w-1 overlaps both. P(w-2) aliases S buffer (w & 1), so S(w) must follow PV(w-2) in the
// (in-order) tensor pipe, which this order guarantees.
template <bool kLog, bool kFull>
__device__ void mma_issuer(const FwdParams& p, Ctl* ctl, uint32_t smem_base, uint32_t tmem,
                           int lane) {
  Ring ring;
  uint32_t q_phase = 0, n_started[2] = {0, 0};
  uint32_t wg = 0;                       // global unit counter
  uint32_t nt[2] = {0, 0};               // units issued so far per tile (barrier selection)
  int sched_n = 0;
  Pend pd0{}, pd1{};                     // FIFO: pd0 older
  int npend = 0;
  auto bar = [&](const void* b) { return smem_u32(b); };
  IT_TRACE_DECL

  // P arrives in two pieces (p_full + 8 c): the MMAs of a piece are issued as soon as it is in TMEM
  auto issue_pend = [&](const Pend& u) {
    IT_TR(0);
    if (u.o_free) mbar_wait(u.o_free, u.ofree_par, 12);
    mbar_wait(u.v_full, u.vphase, 15);
    IT_TR(3);
    mbar_wait(u.p_full, u.par, 13);
    tc_fence_after();
    IT_TR(1);
    mma_ts_e4<8, 128>(u.tmem_o, u.tmem_p, u.vdesc, kIdescPV, u.acc);
    IT_TR(6);
    mbar_wait(u.p_full + 8, u.par, 13);
    tc_fence_after();
    IT_TR(1);
    mma_ts_e4<8, 128>(u.tmem_o, u.tmem_p + 32, u.vdesc + 4 * 128, kIdescPV, 1u);
    tc_commit_e(u.pv_done);
    if (u.v_empty) tc_commit_e(u.v_empty);
    if (u.o_full) tc_commit_e(u.o_full);
    IT_TR(6);
  };
  auto pop = [&]() {
    issue_pend(pd0);
    pd0 = pd1;
    --npend;
  };

  for (;;) {
    const int ss = sched_n % kSched;
    IT_TR(0);
    mbar_wait(smem_u32(&ctl->sched_full[ss]), (sched_n / kSched) & 1, 10);
    IT_TR(4);
    // warp-uniform by construction; the reduction tells the compiler so (see uni())
    int4 item;
    item.x = static_cast<int>(uni(static_cast<uint32_t>(ctl->sched_item[ss].x)));
    item.y = static_cast<int>(uni(static_cast<uint32_t>(ctl->sched_item[ss].y)));
    item.z = static_cast<int>(uni(static_cast<uint32_t>(ctl->sched_item[ss].z)));
    item.w = 0;
    __syncwarp();
    if (lane == 0) mbar_arrive(smem_u32(&ctl->sched_empty[ss]));
    ++sched_n;
    if (item.x < 0) break;
    const ItemT<kFull> it = decode_item<kFull>(p, item);

    RowWalk rw;
    uint32_t rem[2] = {0, 0};            // units each tile still has in this item
    for (int base = 0; base < p.W; base += 64) {
      uint32_t n0, n1;
      rw.load(p, it, base, lane);
      rw.counts(n0, n1);
      rem[0] += n0;
      rem[1] += n1;
    }
    bool first[2] = {true, true};
    [[maybe_unused]] int n_logged = 0;

    // The next Q tiles are loaded only after every softmax warp has read the current ones (row
    // norms), and a softmax warp may be waiting for o_full of a unit still parked in the FIFO: if Q
    // is not there yet, issue the parked PVs first (they need nothing from the next item).
    if (!mbar_try_wait(smem_u32(&ctl->q_full), q_phase))
      while (npend > 0) pop();
    IT_TR(0);
    mbar_wait(smem_u32(&ctl->q_full), q_phase, 11);
    IT_TR(4);
    q_phase ^= 1u;
    tc_fence_after();
    // Key blocks of the union, one ahead: the next block's bookkeeping (mask walk, ring slots,
    // descriptors) is done right after the first half of the current block's last S has been
    // issued, i.e. while the tensor pipe still has those MMAs queued, not between two units.
    struct Blk {
      int j;                             // key block
      bool valid, has0, has1;
      uint32_t k_full, kphase, k_empty, v_full, vphase, v_empty;
      uint64_t kdesc, vdesc;
    };
    int bw = -1;                         // word index of the walk
    uint32_t bx = 0, bx0 = 0, bx1 = 0;   // bits left in the word, the two rows' words
    auto next_blk = [&]() {
      Blk b;
      b.valid = false;
      while (bx == 0u) {
        if (++bw >= p.W) return b;
        if ((bw & 63) == 0 && (bw > 0 || p.W > 64)) rw.load(p, it, bw, lane);
        bx0 = rw.row0(bw);
        bx1 = rw.row1(bw);
        bx = bx0 | bx1;
      }
      const int bit = __ffs(bx) - 1;
      bx &= bx - 1u;
      b.valid = true;
      b.j = bw * 32 + bit;
      b.has0 = ((bx0 >> bit) & 1u) != 0;
      b.has1 = ((bx1 >> bit) & 1u) != 0;
      const int kslot = ring.slot;
      b.kphase = ring.phase;
      ring.advance();
      const int vslot = ring.slot;
      b.vphase = ring.phase;
      ring.advance();
      b.k_full = bar(&ctl->kv_full[kslot]);
      b.k_empty = bar(&ctl->kv_empty[kslot]);
      b.v_full = bar(&ctl->kv_full[vslot]);
      b.v_empty = bar(&ctl->kv_empty[vslot]);
      b.kdesc = make_desc(kDescKMajor, smem_base + kOffRing + kslot * kTileBytes);
      b.vdesc = make_desc(kDescMNMajor, smem_base + kOffRing + vslot * kTileBytes);
      return b;
    };
    Blk cb = next_blk();
    while (cb.valid) {
      Blk nb;
      nb.valid = false;
      bool k_ready = false;
#pragma unroll
      for (int t = 0; t < 2; ++t) {
        if (!(t == 0 ? cb.has0 : cb.has1)) continue;
        const bool last_of_blk = t == 1 || !cb.has1;
        // everything the unit needs, before the issuer blocks on the oldest unit's P
        Pend u;
        const uint32_t buf = wg & 1u, sel = nt[t] & 1u;
        u.tmem_o = tmem + 256 + t * 128;
        u.tmem_p = tmem + buf * 128;
        u.vdesc = cb.vdesc;
        u.acc = first[t] ? 0u : 1u;
        u.p_full = bar(&ctl->p_full[t][sel][0]);
        u.par = (nt[t] >> 1) & 1u;
        u.pv_done = bar(&ctl->pv_done[t][sel]);
        u.v_full = cb.v_full;
        u.vphase = cb.vphase;
        u.o_free = first[t] ? bar(&ctl->o_free[t]) : 0u;
        u.ofree_par = (n_started[t] & 1u) ^ 1u;
        u.v_empty = last_of_blk ? cb.v_empty : 0u;
        u.o_full = (--rem[t] == 0u) ? bar(&ctl->o_full[t]) : 0u;
        const uint32_t tmem_s = tmem + buf * 128;
        const uint64_t qdesc = make_desc(kDescKMajor, smem_base + kOffQ + (it.split() ? 0 : t) * kTileBytes);
        const uint32_t s_full = bar(&ctl->s_full[t][sel]);
        if constexpr (kLog) {          // debug build of the kernel (sa_debug_fwd_walk): the issue order
          if (lane == 0) WalkLog(p).is_seq(it.bh * p.NQB + it.ua)[n_logged] = (t << 15) | cb.j;
          ++n_logged;
        }
        ++nt[t];
        if (first[t]) ++n_started[t];
        first[t] = false;
        ++wg;
        IT_TR(0);
        if (!k_ready) k_ready = mbar_try_wait(cb.k_full, cb.kphase);
        IT_TR(2);
        if (npend == 2) pop();           // PV of the oldest unit: it frees this unit's S buffer
        if (!k_ready) {
          IT_TR(0);
          mbar_wait(cb.k_full, cb.kphase, 14);
          IT_TR(2);
          k_ready = true;
        }
        tc_fence_after();
        IT_TR(0);
        mma_ss_e4<2, 2>(tmem_s, qdesc, cb.kdesc, kIdescQK, 0u);
        if (last_of_blk) nb = next_blk();
        mma_ss_e4<2, 2>(tmem_s, qdesc + (kHalfBytes >> 4), cb.kdesc + (kHalfBytes >> 4), kIdescQK, 1u);
        tc_commit_e(s_full);
        IT_TR(5);
        IT_TRACE_UNIT
        if (npend == 0) pd0 = u; else pd1 = u;
        ++npend;
      }
      tc_commit_e(cb.k_empty);
      cb = nb;
    }
    if constexpr (kLog) {
      if (lane == 0) WalkLog(p).is_cnt()[it.bh * p.NQB + it.ua] = n_logged;
    }
    tc_commit_e(smem_u32(&ctl->q_empty));   // every S of this item has been issued
    // No S can follow until the next item's Q tiles have arrived, and their load starts only now:
    // issue the older parked PV at once (the younger one's P is still being computed; it goes out
    // after the next item's bookkeeping, see above).
    if (npend == 2) pop();
  }
  while (npend > 0) pop();
  IT_TRACE_REPORT
}

// P = 2^(c*s - m) of one query row (128 columns in sr), written to TMEM as bf16 in kPChunks pieces
// (p_full[piece] arrives after each); returns the row sum. Packed FFMA2 for the argument; of every
// 4 column pairs NPOLY take the FMA-pipe exp2 and the rest MUFU.EX2 (the ragged tile uses
// NPOLY = 0: MUFU turns its -inf columns into an exact 0). Row sum in 4 packed accumulators.
template <int NPOLY>
__device__ __forceinline__ float exp_tile(const uint32_t (&sr)[4][32], float c, float m_use,
                                          uint32_t tm_p, uint64_t* p_full, int lane) {
  const uint64_t c2 = pk2(c, c), nm2 = pk2(-m_use, -m_use);
  uint64_t lacc[4] = {0ull, 0ull, 0ull, 0ull};
#pragma unroll
  for (int cc = 0; cc < 4; ++cc) {
    uint32_t pk[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
      const uint64_t x = fma2(pk2(__uint_as_float(sr[cc][2 * i]), __uint_as_float(sr[cc][2 * i + 1])),
                              c2, nm2);
      float p0, p1;
      if ((i & 3) < NPOLY) {
        exp2_fma_pipe(x, p0, p1);
      } else {
        float x0, x1;
        up2(x, x0, x1);
        p0 = ex2(x0);
        p1 = ex2(x1);
      }
      lacc[i & 3] = add2(lacc[i & 3], pk2(p0, p1));
      pk[i] = pack_bf16x2(p0, p1);
    }
    // The arrival for a piece is deferred until the next piece's exponentials are in registers:
    // by then its tcgen05.st has long completed and wait::st does not stall.
    constexpr int kPer = 4 / kPChunks;
    if (cc % kPer == 0 && cc > 0) {
      tc_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&p_full[cc / kPer - 1]));
    }
    tmem_st16(tm_p + cc * 16, pk);
  }
  tc_wait_st();
  tc_fence_before();
  __syncwarp();
  if (lane == 0) mbar_arrive(smem_u32(&p_full[kPChunks - 1]));
  float a0, a1, b0, b1;
  up2(add2(lacc[0], lacc[1]), a0, a1);
  up2(add2(lacc[2], lacc[3]), b0, b1);
  return (a0 + a1) + (b0 + b1);
}

// ------------------------------------------------------------------ warps 4-11: softmax + epilogue
// One thread per query row: thread (quarter, lane) of warpgroup t owns TMEM lane 32*quarter+lane
// of S_t / O_t, so row max and row sum need no shuffles.
template <bool kLog, bool kFull>
__device__ void softmax_wg(const FwdParams& p, Ctl* ctl, uint32_t smem_base, uint32_t tmem, int t,
                           int quarter, int lane) {
  const int row = quarter * 32 + lane;
  const uint32_t lane_base = static_cast<uint32_t>(quarter * 32) << 16;
  const uint32_t tm_o = tmem + lane_base + 256 + t * 128;
  const float c = p.scale_log2;
  const bool out32 = (reinterpret_cast<uintptr_t>(p.out) & 31u) == 0;   // rows are 256 B apart
  uint32_t o_phase = 0, qf_phase = 0;
  uint32_t wg = 0;                       // global unit counter, in step with the MMA issuer
  uint32_t nmine = 0;                    // this tile's units so far (barrier selection: every phase
                                         // of s_full[t][.] is consumed in order, none is skipped)
  int sched_n = 0;
  uint32_t n_fixed = 0, n_exact = 0;     // items of this warp by softmax path (p.stats)
  uint32_t n_split = 0;                  // split items so far (parity of the xchg barriers)
  SA_TRACE_DECL
  // Per item: what the walk needs (the item, its bit-rows, the rows' score bound). next_item() takes
  // the next item from the scheduler ring and waits for its Q tiles; it is called for item n+1
  // BEFORE the epilogue of item n, so that the wait for the Q tiles and the row norms fall into the
  // time this warpgroup would otherwise spend waiting for the last PV of item n.
  ItemT<kFull> it{};
  bool exists = false;
  RowWalk rw;
  float bound = 0.f;
  auto next_item = [&]() {
    const int ss = sched_n % kSched;
    SA_TR(0);
    mbar_wait(smem_u32(&ctl->sched_full[ss]), (sched_n / kSched) & 1, 20);
    SA_TR(5);
    const int4 item = ctl->sched_item[ss];
    __syncwarp();
    if (lane == 0) mbar_arrive(smem_u32(&ctl->sched_empty[ss]));
    ++sched_n;
    if (item.x < 0) return false;
    it = decode_item<kFull>(p, item);
    exists = t == 0 || it.has1;   // tile 1 is empty in single-row items and past the last row

    // An upper bound of every score of this query row (Cauchy-Schwarz): scale * |q_i| * max_j |k_j|,
    // in the log2 domain. |q_i| comes from the Q tile in shared memory (128B-swizzled rows), max |k|
    // from the pre-pass. If the first key block shows that the bound is not far above the real
    // scores, it becomes the row's softmax reference point for the whole item: no running max, no
    // rescale, and the row-max pass (a third of the softmax instructions) disappears. Otherwise the
    // warp keeps the exact running max. Either way the result is the same softmax.
    rw.load(p, it, 0, lane);
    const float kmax2 = p.kmax2 ? __ldg(p.kmax2 + it.bh) : 0.f;   // in flight while Q arrives
    SA_TR(0);
    mbar_wait(smem_u32(&ctl->q_full), qf_phase, 24);
    SA_TR(6);
    qf_phase ^= 1u;
    bound = INFINITY;                    // no bound (sparse group / small problem): exact running max,
    if (exists && p.kmax2 != nullptr && kmax2 >= 0.f) {      // and the row norms are not needed
      const uint32_t qrow = smem_base + kOffQ + (it.split() ? 0 : t) * kTileBytes + row * 128;
      float qn2 = 0.f;
#pragma unroll
      for (int ch = 0; ch < 16; ++ch) {
        const uint32_t addr = qrow + (ch >> 3) * kHalfBytes + (((ch & 7) ^ (row & 7)) << 4);
        uint32_t w0, w1, w2, w3;
        asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(w0), "=r"(w1), "=r"(w2), "=r"(w3) : "r"(addr));
        const uint32_t wv[4] = {w0, w1, w2, w3};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const float lo = __uint_as_float(wv[i] << 16), hi = __uint_as_float(wv[i] & 0xFFFF0000u);
          qn2 = fmaf(lo, lo, qn2);
          qn2 = fmaf(hi, hi, qn2);
        }
      }
      bound = c * sqrtf(qn2) * sqrtf(kmax2);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(smem_u32(&ctl->q_empty));   // this warp is done with the Q tiles
    SA_TR(7);
    return true;
  };

  bool have_item = next_item();
  while (have_item) {
    float m_run = -INFINITY, l_run = 0.f;
    bool started = false;
    bool fixed = false;                  // warp-uniform: m_run is the bound, fixed for the item
    uint32_t prev_unit = 0xFFFFFFFEu;    // this tile's previous unit in the item
    [[maybe_unused]] const uint32_t wg_item0 = wg;
    [[maybe_unused]] int n_logged = 0;
    // Walk this tile's own bit-row. A unit's number in the union walk order (which the MMA issuer
    // follows) is the popcount of both rows below its bit. The next unit's bookkeeping is computed
    // in the same straight-line block as the exponentials, so it does not sit in the cycle
    // S -> softmax -> PV -> next S.
    for (int w = 0; w < p.W; ++w) {
      if ((w & 63) == 0 && w > 0) rw.load(p, it, w, lane);
      const uint32_t x0 = rw.row0(w), x1 = rw.row1(w);
      uint32_t xm = t == 0 ? x0 : x1;
      const uint32_t wbase = wg;
      wg += __popc(x0) + __popc(x1);
      if (!xm) continue;
      int bit = __ffs(xm) - 1;
      xm &= xm - 1u;
      uint32_t my = wbase + __popc(x0 & ((1u << bit) - 1u)) + __popc(x1 & ((1u << bit) - 1u)) +
                    (t == 1 ? (x0 >> bit) & 1u : 0u);
      for (;;) {
        const int j = w * 32 + bit;
        if constexpr (kLog) {
          if (quarter == 0 && lane == 0 && !(t == 1 && it.split()))   // a split item's row: tile 0 logs
            WalkLog(p).wg_seq(static_cast<size_t>(it.bh) * p.NQB + (t == 0 ? it.ua : it.ub))[n_logged] =
                static_cast<int32_t>(((my - wg_item0) << 16) | static_cast<uint32_t>(j));
          ++n_logged;
        }
        const uint32_t buf = my & 1u, sel = nmine & 1u, par = (nmine >> 1) & 1u;
        const uint32_t tm_s = tmem + lane_base + buf * 128;
        SA_TR(0);
        mbar_wait(smem_u32(&ctl->s_full[t][sel]), par, 21);
        tc_fence_after();
        SA_TR(1);
        uint32_t sr[4][32];
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) tmem_ld32(tm_s + cc * 32, sr[cc]);
        tc_wait_ld();
        SA_TR(2);
        // keys >= n_valid carry zero weight (only the ragged tail block can hold any)
        const int kv = p.n_valid - j * kBlk;
        const bool ragged = kv < kBlk;
        if (ragged) {
#pragma unroll
          for (int cc = 0; cc < 4; ++cc)
#pragma unroll
            for (int i = 0; i < 32; ++i)
              if (cc * 32 + i >= kv) sr[cc][i] = 0xFF800000u;   // -inf
        }
        if (!fixed) {
        // row max: four independent chains of 3-input max
        float mxa[4];
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
          mxa[cc] = fmaxf(__uint_as_float(sr[cc][0]), __uint_as_float(sr[cc][1]));
#pragma unroll
          for (int i = 2; i < 32; i += 2)
            mxa[cc] = max3(mxa[cc], __uint_as_float(sr[cc][i]), __uint_as_float(sr[cc][i + 1]));
        }
        const float m_new = max3(fmaxf(mxa[0], mxa[1]), mxa[2], mxa[3]) * c;
        const bool need = m_new > m_run + kRescaleThreshold;   // also true for the first finite max
        if (__any_sync(0xFFFFFFFFu, need)) {
          float alpha = 1.f;
          if (need) {
            alpha = ex2(m_run - m_new);      // m_run = -inf -> 0
            m_run = m_new;
            l_run *= alpha;
          }
          if (started) {                     // O_t holds earlier blocks: bring it to the new max
            // PV(my-2) and older retired before S(my) was issued; PV(my-1) may still be in flight
            if (prev_unit + 1u == my) {
              mbar_wait(smem_u32(&ctl->pv_done[t][(nmine - 1u) & 1u]), ((nmine - 1u) >> 1) & 1u, 23);
              tc_fence_after();
            }
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) {
              uint32_t orr[32];
              tmem_ld32(tm_o + cc * 32, orr);
              tc_wait_ld();
#pragma unroll
              for (int i = 0; i < 32; ++i) orr[i] = __float_as_uint(__uint_as_float(orr[i]) * alpha);
              tmem_st32(tm_o + cc * 32, orr);
            }
          }
        }
        if (!started) {
          // first unit of the item: every row of the warp has a finite maximum and its bound lies
          // at most kBoundSlack above it -> 2^(s*c - bound) cannot underflow for the row's largest
          // scores (the real maximum over the item is at least this block's), and never exceeds 1
          fixed = __all_sync(0xFFFFFFFFu, m_run > -INFINITY && bound <= m_run + kBoundSlack);
          if (fixed) m_run = bound;
          n_fixed += fixed ? 1u : 0u;
          n_exact += fixed ? 0u : 1u;
        }
        }
        const float m_use = (m_run == -INFINITY) ? 0.f : m_run;
        SA_TR(3);
        // this tile's next unit in the word, if any (nbit = -1 -> the values are not used)
        const bool more = xm != 0u;
        const int nbit = (__ffs(xm) - 1) & 31;
        xm &= xm - 1u;
        const uint32_t nmy = wbase + __popc(x0 & ((1u << nbit) - 1u)) + __popc(x1 & ((1u << nbit) - 1u)) +
                             (t == 1 ? (x0 >> nbit) & 1u : 0u);
        if (ragged) l_run += exp_tile<0>(sr, c, m_use, tm_s, ctl->p_full[t][sel], lane);
        else l_run += exp_tile<kPolyPairs>(sr, c, m_use, tm_s, ctl->p_full[t][sel], lane);
        SA_TR(4);
        started = true;
        prev_unit = my;
        ++nmine;
        if (!more) break;
        bit = nbit;
        my = nmy;
      }
    }

    // ---- epilogue: O / l -> bf16, lse = ln2 * (m + log2 l); empty row -> 0 / -inf
    if constexpr (kLog) {
      if (exists && quarter == 0 && lane == 0 && !(t == 1 && it.split())) {
        const size_t lrow = static_cast<size_t>(it.bh) * p.NQB + (t == 0 ? it.ua : it.ub);
        const int partner = t == 0 ? (it.has1 ? it.ub : -1) : it.ua;
        WalkLog(p).wg_cnt()[lrow] = n_logged;
        WalkLog(p).wg_info()[lrow] = ((partner + 1) << 1) | t;
      }
    }
    const bool wrote = exists;
    const bool split = it.split();
    // a part of a row (one key range of it) leaves its normalised O and its lse in scratch slot
    // `part`; combine_parts_kernel (next on the stream) merges the row's parts into out / lse
    const size_t grow = it.part < 0
        ? static_cast<size_t>(it.row0) + static_cast<size_t>(t == 0 ? it.ua : it.ub) * kBlk + row
        : static_cast<size_t>(2 * it.part + (split ? 0 : t)) * kBlk + row;
    uint4* orow = reinterpret_cast<uint4*>((it.part < 0 ? p.out : p.part_out) + grow * kD);
    float* lrow = (it.part < 0 ? p.lse : p.part_lse) + grow;
    // (the epilogue comes BEFORE the next item is taken up: the next item's Q tiles are in flight
    // meanwhile, so the wait for them, ~1000 clk when taken first, is gone: +0.3-2% at every size)
    do {
    if (!wrote) break;
    if (split) {
      // ---- a split item: the two warpgroups hold the two halves (even / odd key blocks) of ONE query
      // block, each with its own running maximum, row sum and O tile. Warpgroup 1 publishes (m, l) of
      // its half -- in the first 8 bytes of the output row, which warpgroup 0 overwrites afterwards --
      // and leaves its O tile in TMEM; warpgroup 0 (same TMEM lanes) reads both tiles, 32 columns at a
      // time (no more live registers than the plain epilogue: the per-block loop has none to spare), and
      // writes  out = (O0 2^(m0-M) + O1 2^(m1-M)) / (l0 2^(m0-M) + l1 2^(m1-M)),  lse = ln2 (M + log2(.)),
      // M = max(m0, m1): the same softmax, summed in a fixed order (deterministic).
      float2* xchg = reinterpret_cast<float2*>(orow);
      if (started) {
        mbar_wait(smem_u32(&ctl->o_full[t]), o_phase, 22);     // this half's O tile is complete
        o_phase ^= 1u;
      }
      // (hand-off through an mbarrier pair with back-pressure: a half without units publishes at once,
      // and must not get two items ahead of the reader)
      if (t == 1) {
        mbar_wait(smem_u32(&ctl->xchg_empty), (n_split & 1u) ^ 1u, 26);
        __stcg(xchg, make_float2(started ? m_run : -INFINITY, started ? l_run : -1.f));   // l < 0: no units
        __threadfence_block();
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctl->xchg_full));
        ++n_split;
        break;                             // O1 is released by warpgroup 0 once it has read it
      }
      mbar_wait(smem_u32(&ctl->xchg_full), n_split & 1u, 27);
      ++n_split;
      tc_fence_after();
      float2 ml1 = __ldcg(xchg);
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctl->xchg_empty));
      const bool other = ml1.y >= 0.f;     // tile 1 had units in this item: its O tile is valid
      ml1.y = fmaxf(ml1.y, 0.f);
      const float m0 = started ? m_run : -INFINITY, l0 = started ? l_run : 0.f;
      const float M = fmaxf(m0, ml1.x);
      const float a0 = m0 > -INFINITY ? ex2(m0 - M) : 0.f, a1 = ml1.x > -INFINITY ? ex2(ml1.x - M) : 0.f;
      const float L = l0 * a0 + ml1.y * a1;
      const float inv = L > 0.f ? 1.f / L : 0.f;
      const float s0 = started ? a0 * inv : 0.f, s1 = other ? a1 * inv : 0.f;
#pragma unroll 1
      for (int cc = 0; cc < 4; ++cc) {
        uint32_t o0[32], o1[32];
        tmem_ld32(tm_o + cc * 32, o0);                 // (an unused tile's columns hold old finite data or
        tmem_ld32(tm_o + 128 + cc * 32, o1);           //  anything at all: its weight below is exactly 0)
        tc_wait_ld();
#pragma unroll
        for (int ch = 0; ch < 4; ++ch) {
          uint32_t v[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const int i = 8 * ch + 2 * k;
            const float x0 = s0 != 0.f ? __uint_as_float(o0[i]) * s0 : 0.f;
            const float x1 = s0 != 0.f ? __uint_as_float(o0[i + 1]) * s0 : 0.f;
            const float y0 = s1 != 0.f ? fmaf(__uint_as_float(o1[i]), s1, x0) : x0;
            const float y1 = s1 != 0.f ? fmaf(__uint_as_float(o1[i + 1]), s1, x1) : x1;
            v[k] = pack_bf16x2(y0, y1);
          }
          orow[cc * 4 + ch] = make_uint4(v[0], v[1], v[2], v[3]);
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (started) mbar_arrive(smem_u32(&ctl->o_free[0]));
        if (other) mbar_arrive(smem_u32(&ctl->o_free[1]));
      }
      *lrow = L > 0.f ? 0.6931471805599453f * (M + lg2(L)) : -INFINITY;
    } else if (started) {
      SA_TR(0);
      mbar_wait(smem_u32(&ctl->o_full[t]), o_phase, 22);
      SA_TR(8);
      o_phase ^= 1u;
      tc_fence_after();
      const float inv = l_run > 0.f ? 1.f / l_run : 0.f;
      // the whole row of O to registers first (the S registers are dead here), O_t released to the
      // next item's first PV before the conversion and the stores
      uint32_t orr[4][32];
#pragma unroll
      for (int cc = 0; cc < 4; ++cc) tmem_ld32(tm_o + cc * 32, orr[cc]);
      tc_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctl->o_free[t]));
#pragma unroll
      for (int cc = 0; cc < 4; ++cc) {
        // 32 columns -> 64 B of the row: two 256-bit stores, a full 32 B sector per lane each
        // (four 128-bit stores if the caller's out is only 16 B aligned, which the ABI allows)
#pragma unroll
        for (int i = 0; i < 2; ++i) {
          uint32_t v[8];
#pragma unroll
          for (int k = 0; k < 8; ++k)
            v[k] = pack_bf16x2(__uint_as_float(orr[cc][16 * i + 2 * k]) * inv,
                               __uint_as_float(orr[cc][16 * i + 2 * k + 1]) * inv);
          if (out32) {
            st_global_256(orow + cc * 4 + i * 2, v);
          } else {
            orow[cc * 4 + i * 2] = make_uint4(v[0], v[1], v[2], v[3]);
            orow[cc * 4 + i * 2 + 1] = make_uint4(v[4], v[5], v[6], v[7]);
          }
        }
      }
      *lrow = l_run > 0.f ? 0.6931471805599453f * (m_run + lg2(l_run)) : -INFINITY;
      SA_TR(9);
      SA_TRACE_ITEM
    } else {
      const uint4 z = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
      for (int i = 0; i < 16; ++i) orow[i] = z;
      *lrow = -INFINITY;
    }
    } while (false);
    have_item = next_item();             // (overwrites it, exists, rw, bound)
  }
  if (p.stats != nullptr && lane == 0) {
    atomicAdd(p.stats, static_cast<int32_t>(n_fixed));
    atomicAdd(p.stats + 1, static_cast<int32_t>(n_exact));
  }
  SA_TRACE_REPORT
}

// ------------------------------------------------------------------ kernel
template <bool kLog, bool kFull>
__global__ void __launch_bounds__(kThreads, 1)
fwd_tcgen05_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                   const __grid_constant__ CUtensorMap tm_v, const FwdParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t smem_base = (raw + 1023u) & ~1023u;
  Ctl* ctl = reinterpret_cast<Ctl*>(smem_raw + (smem_base - raw) + kOffCtl);
  // warp index through a shuffle: the compiler then knows it is warp-uniform, and so is the role branch
  const int warp = __shfl_sync(0xFFFFFFFFu, static_cast<int>(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    prefetch_tensormap(&tm_q);
    prefetch_tensormap(&tm_k);
    prefetch_tensormap(&tm_v);
    mbar_init(smem_u32(&ctl->q_full), 1);
    mbar_init(smem_u32(&ctl->q_empty), 1 + 8);   // MMA commit + the 8 softmax warps (row norms)
    for (int s = 0; s < kSlots; ++s) {
      mbar_init(smem_u32(&ctl->kv_full[s]), 1);
      mbar_init(smem_u32(&ctl->kv_empty[s]), 1);
    }
    for (int t = 0; t < 2; ++t) {
      for (int b = 0; b < 2; ++b) {
        mbar_init(smem_u32(&ctl->s_full[t][b]), 1);
        mbar_init(smem_u32(&ctl->pv_done[t][b]), 1);
        for (int c = 0; c < 4; ++c)
          mbar_init(smem_u32(&ctl->p_full[t][b][c]), 4);   // one arrival per softmax warp
      }
      mbar_init(smem_u32(&ctl->o_full[t]), 1);
      mbar_init(smem_u32(&ctl->o_free[t]), 4);
      if (t == 0) {
        mbar_init(smem_u32(&ctl->xchg_full), 4);     // one arrival per warp of warpgroup 1
        mbar_init(smem_u32(&ctl->xchg_empty), 4);    // one arrival per warp of warpgroup 0
      }
    }
    for (int s = 0; s < kSched; ++s) {
      mbar_init(smem_u32(&ctl->sched_full[s]), 1);
      mbar_init(smem_u32(&ctl->sched_empty[s]), 9);  // MMA thread + 8 softmax warps
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
  griddep_wait();      // barriers, TMEM and tensor maps were set up under the pre-pass's tail

  if (warp < 4) {
    setmaxnreg_dec<88>();
    if (warp == 0) {
      producer<kFull>(p, ctl, smem_base, &tm_q, &tm_k, &tm_v, lane);
    } else if (warp == 1) {
      mma_issuer<kLog, kFull>(p, ctl, smem_base, tmem, lane);
    }
  } else {
    setmaxnreg_inc<208>();
    softmax_wg<kLog, kFull>(p, ctl, smem_base, tmem, warp >= 8 ? 1 : 0, warp & 3, lane);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem, kTmemCols);
}

// ------------------------------------------------------------------ host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      f = nullptr;
    return reinterpret_cast<EncodeTiledFn>(f);
  }();
  return fn;
}

// [rows][128] bf16 row-major viewed as a 2-D tensor; box = 64 columns x 128 rows, 128B swizzle
bool make_map(CUtensorMap* m, const void* base, uint64_t rows) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t gdim[2] = {static_cast<cuuint64_t>(kD), rows};
  const cuuint64_t gstride[1] = {static_cast<cuuint64_t>(kD) * 2};
  const cuuint32_t box[2] = {64, static_cast<cuuint32_t>(kBlk)};
  const cuuint32_t estr[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), gdim, gstride, box,
            estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

// shared with sig_tcgen05.cu: CUtensorMap of a [rows][128] bf16 array, box 64 x 128, 128B swizzle
bool make_tile_map_128x64(void* map, const void* base, uint64_t rows) {
  return make_map(static_cast<CUtensorMap*>(map), base, rows);
}

cudaError_t launch_fwd_tcgen05(const FwdParams& p, void*, cudaStream_t st, int* n_launch,
                               const char** err_text) {
  int n_sm = 0;
  cudaError_t e = device_sm_count(&n_sm);
  if (e != cudaSuccess) return e;
  const bool log = p.walk_log != nullptr;
  const bool lean = !log && p.lean_items;        // the work list holds neither split items nor parts
  e = log ? ensure_dynamic_smem(kSmemFwdTcgen05Log, reinterpret_cast<const void*>(fwd_tcgen05_kernel<true, true>),
                                static_cast<int>(kSmemBytes))
          : lean ? ensure_dynamic_smem(kSmemFwdTcgen05Lean,
                                       reinterpret_cast<const void*>(fwd_tcgen05_kernel<false, false>),
                                       static_cast<int>(kSmemBytes))
                 : ensure_dynamic_smem(kSmemFwdTcgen05, reinterpret_cast<const void*>(fwd_tcgen05_kernel<false, true>),
                                       static_cast<int>(kSmemBytes));
  if (e != cudaSuccess) { *err_text = "cudaFuncSetAttribute(fwd_tcgen05_kernel)"; return e; }
  CUtensorMap tq, tk, tv;
  const uint64_t rows = static_cast<uint64_t>(p.B) * p.H * p.N;
  if (!make_map(&tq, p.q, rows) || !make_map(&tk, p.k, rows) || !make_map(&tv, p.v, rows)) {
    *err_text = "cuTensorMapEncodeTiled failed";
    return cudaErrorInvalidValue;
  }
  const int grid = p.n_items < n_sm ? p.n_items : n_sm;   // n_items: upper bound (pairs are mask-dependent)
  e = log ? launch_pdl(fwd_tcgen05_kernel<true, true>, dim3(grid), dim3(kThreads), kSmemBytes, st, tq, tk, tv, p)
          : lean ? launch_pdl(fwd_tcgen05_kernel<false, false>, dim3(grid), dim3(kThreads), kSmemBytes, st, tq, tk,
                              tv, p)
                 : launch_pdl(fwd_tcgen05_kernel<false, true>, dim3(grid), dim3(kThreads), kSmemBytes, st, tq, tk,
                              tv, p);
  if (e != cudaSuccess) return e;
  *n_launch += 1;
  return cudaGetLastError();
}

}  // namespace sa

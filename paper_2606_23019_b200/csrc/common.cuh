// common.cuh -- shared declarations of the CUDA library (product side only; the oracle never
// includes this).
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/scalingattn.h"

namespace sa {

// ---- CRM forward iterator (App. E Alg. 2), one instance per walking thread ----
// State {ptr, end, val, base} as in the paper. INIT sets base = -32 and prefetches the first
// non-zero word; ADVANCE skips zero words (base += 32 per word); INDEX = base + CTZ(val), here
// __ffs(val) - 1; NEXT clears the lowest set bit (val &= val - 1). The last word is ANDed with the
// valid-bit mask so stray bits at positions >= NKB cannot index past the last key block.
struct CrmIter {
  const uint32_t* ptr;
  const uint32_t* end;
  uint32_t val;
  uint32_t tail_mask;
  int base;

  __device__ __forceinline__ void advance() {
    while (val == 0u && ptr != end) {
      val = __ldg(ptr);
      ++ptr;
      if (ptr == end) val &= tail_mask;
      base += 32;
    }
  }
  __device__ __forceinline__ void init(const uint32_t* row_ptr, int n_words, int nkb) {
    ptr = row_ptr;
    end = row_ptr + n_words;
    val = 0u;
    base = -32;
    tail_mask = (nkb & 31) ? ((1u << (nkb & 31)) - 1u) : 0xFFFFFFFFu;
    advance();
  }
  // -1 is the end-of-row sentinel
  __device__ __forceinline__ int index() const { return val ? base + (__ffs(val) - 1) : -1; }
  __device__ __forceinline__ void next() {
    val &= val - 1u;
    if (val == 0u) advance();
  }
};

// ---- forward-pass problem description handed to the kernels ----
struct FwdParams {
  const __nv_bfloat16* q;
  const __nv_bfloat16* k;
  const __nv_bfloat16* v;
  const uint32_t* mask_bits;
  __nv_bfloat16* out;
  float* lse;
  int B, H, N, n_valid, D, Bq, Bk;
  int NQB, NKB, W;
  float scale;
  float scale_log2;   // scale * log2(e)
  // schedule (workspace)
  const int4* items;          // work items in issue order: x = b*H + h, y = ua | ub << 16 (query blocks
                              // of the item; ub = 0xFFFF: single-row item), z = scratch slot of a
                              // part (-1: whole rows)
  const uint32_t* part_mask;  // parts of rows: [slot][tile][W] the bit-rows restricted to the part's key range
  __nv_bfloat16* part_out;    // parts of rows (tcgen05 kernel): [slot][tile][128][D] normalised O
  float* part_lse;            //                                  [slot][tile][128] lse of the part
  const int32_t* n_items_dev; // number of work items, written by the pre-pass (pair items: mask-dependent)
  int32_t* counter;           // dynamic scheduler cursor (zeroed by the pre-pass)
  const float* kmax2;         // [B*H] max |k|^2 over the valid keys (tcgen05 kernel only)
  int n_items;                // host-side count: exact for single-row items, an upper bound for pairs
  int rows_per_item;          // query blocks per work item: 2 (a pair shares its K/V tiles) or 1
  int split_rows;             // single-row items are split items (tcgen05 kernel): see Item::split
  int lean_items;             // the work list holds no split item and no part: the lean kernel build runs it
  int32_t* stats;             // [2] (warp, item) counts by softmax path: fixed reference point / exact
                              // running max (zeroed by the pre-pass; tcgen05 kernel only)
  int32_t* walk_log;          // sa_debug_fwd_walk only (else null): see WalkLog in fwd_tcgen05.cu
};

// Workspace layout for the forward pass (int32 words):
//   [0]                  scheduler cursor
//   [1]                  number of work items
//   [2], [3]             (warp, item) counts of the last tcgen05 call by softmax path (fixed / exact)
//   [16 .. 16+BH)        per-(b,h) total cost (active tiles)
//   [.. + BH)            per-(b,h) number of items
//   [.. + BH)            fp32: per (b,h) max over the valid keys of |k|^2
//   [.. + BH)            per-(b,h) number of items at the tail of the issue order
//   int4 [BH*NQB]        per-(b,h) items, cost descending: {cost, ua | ub << 16, part slot or -1, 0}
//   int4 [BH*NQB]        all items in issue order: {b*H + h, ua | ub << 16, part slot or -1, 0}
//   int4 [rem]           rows issued in parts: {b*H + h (-1: not split after all), ua | ub << 16, parts, first slot}
//   uint32               [rem * parts][2][W] the parts' bit-rows (the rows' bits inside the part's key range)
//   bf16 / fp32          part results: [rem * parts][2][128][128] O and [rem * parts][2][128] lse
// TailPlan: the last, partly filled round of pair items over the SMs is cut into key ranges: `rem`
// pairs (spread over the (b,h) groups, each group's lightest) are issued in `parts` parts each.
struct TailPlan {
  int rem = 0, parts = 0;
};
TailPlan fwd_tail_plan(int B, int H, int NQB, int NKB, int n_sm);
struct FwdWorkspace {
  int32_t* cursor;
  int32_t* n_items;
  int32_t* stats;
  int32_t* head_cost;
  int32_t* head_count;
  int32_t* head_tail;         // [B*H] how many of the group's items go to the tail of the issue order
  float* kmax2;               // [B*H] max over valid keys of |k|^2
  int4* local_items;
  int4* items;
  int4* tasks;                // [plan.rem] rows issued in parts
  uint32_t* part_mask;
  __nv_bfloat16* part_out;
  float* part_lse;
};
size_t fwd_workspace_bytes(int B, int H, int NQB, int W, TailPlan plan);
FwdWorkspace carve_fwd_workspace(void* ws, int B, int H, int NQB, int W, TailPlan plan);

// per-device state (device.cu): SM count of the current device; dynamic shared-memory opt-in of a
// kernel, set once per (device, kernel)
enum SmemKernel { kSmemFwdTcgen05 = 0, kSmemFwdTcgen05Lean, kSmemFwdTcgen05Log, kSmemSigTcgen05, kSmemScheduleItems, kSmemFwdMmaSync64,
                  kSmemFwdMmaSync128, kSmemMaskFromThreshold, kSmemL2Fill, kNumSmemKernels };
cudaError_t device_sm_count(int* n_sm);
// static_scratch.cu: device address and size of the library's fixed scratch array on the current device
cudaError_t static_scratch(void** ptr, size_t* bytes);
cudaError_t ensure_dynamic_smem(SmemKernel id, const void* func, int bytes);

// Programmatic dependent launch: the kernel may be scheduled while its predecessor on the stream is
// still running (its launch latency and prologue overlap the predecessor's tail); it must execute
// griddep_wait() before it reads anything the predecessor (or anything before that) wrote.
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                              Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
#ifdef SA_NO_PDL
  cfg.numAttrs = 0;
#else
  cfg.numAttrs = 1;
#endif
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// launchers (each returns the cudaError_t of its launches; *n_launch += kernels enqueued)
cudaError_t launch_schedule(const FwdParams& p, const FwdWorkspace& w, int rows_per_item,
                            TailPlan plan, cudaStream_t st, int* n_launch, bool reuse = false);
cudaError_t launch_combine_parts(const FwdParams& p, const FwdWorkspace& w, TailPlan plan,
                                 cudaStream_t st, int* n_launch);
cudaError_t launch_fwd_mma_sync(const FwdParams& p, cudaStream_t st, int* n_launch);
cudaError_t launch_fwd_tcgen05(const FwdParams& p, void* ws_extra, cudaStream_t st, int* n_launch,
                               const char** err_text);
cudaError_t launch_pack_mask(const float* scores, const float* density, uint32_t* mask_bits, int H,
                             int NQB, int NKB, int force_diag, void* ws, cudaStream_t st);
size_t pack_mask_workspace_bytes(int H, int NQB, int NKB);
constexpr int kPackMaskLaunches = 5;   // kernels launch_pack_mask enqueues (plus one memset)
cudaError_t launch_mask_from_threshold(const float* tmap, const float* p_star, uint32_t* mask_bits,
                                       int H, int nbq, int nbk, int NQB, int NKB, int force_diag,
                                       cudaStream_t st);
bool make_tile_map_128x64(void* map /* CUtensorMap* */, const void* base, uint64_t rows);
cudaError_t launch_block_significance(const __nv_bfloat16* q, const __nv_bfloat16* k, const float* lse,
                                      float* sig, int B, int H, int N, int n_valid, float scale,
                                      cudaStream_t st, const char** err_text);
size_t threshold_update_workspace_bytes(int B, int H, int NQB, int NKB);
constexpr int kMaxThresholdLevels = 256;
cudaError_t launch_threshold_update(const float* sig, const float* levels, int n_levels, float* tmap,
                                    int B, int H, int NQB, int NKB, void* ws, cudaStream_t st,
                                    int* n_launch);
cudaError_t launch_fidelity(const float* lse_dense, const float* lse_sparse, const int32_t* rows,
                            int n_rows, int BH, int N, float* fidelity, float* per_row,
                            cudaStream_t st);
cudaError_t launch_ex2_rate(int iters, float* sink, int n_sm, cudaStream_t st, double* n_exp);
cudaError_t launch_l2_fill(const void* buf, size_t buf_bytes, int iters, int n_sm, cudaStream_t st,
                           double* bytes_moved);
cudaError_t launch_enumerate(const uint32_t* mask_bits, int H, int NQB, int NKB, int32_t* idx,
                             int32_t* cnt, cudaStream_t st);

}  // namespace sa

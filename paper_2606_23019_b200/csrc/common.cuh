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
  const int2* items;          // work items in issue order: x = b*H + h, y = ua | ub << 16 (query blocks
                              // of the item; ub = 0xFFFF: single-row item)
  const int32_t* n_items_dev; // number of work items, written by the pre-pass (pair items: mask-dependent)
  int32_t* counter;           // dynamic scheduler cursor (zeroed by the pre-pass)
  const float* kmax2;         // [B*H] max |k|^2 over the valid keys (tcgen05 kernel only)
  int n_items;                // host-side count: exact for single-row items, an upper bound for pairs
  int rows_per_item;          // query blocks per work item: 2 (a pair shares its K/V tiles) or 1
  int split_rows;             // single-row items are split items (tcgen05 kernel): see Item::split
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
//   int2 [BH*NQB]        per-(b,h) items, cost descending: {cost, ua | ub << 16}
//   int2 [BH*NQB]        all items in issue order: {b*H + h, ua | ub << 16}
struct FwdWorkspace {
  int32_t* cursor;
  int32_t* n_items;
  int32_t* stats;
  int32_t* head_cost;
  int32_t* head_count;
  float* kmax2;               // [B*H] max over valid keys of |k|^2
  int2* local_items;
  int2* items;
};
size_t fwd_workspace_bytes(int B, int H, int NQB);
FwdWorkspace carve_fwd_workspace(void* ws, int B, int H, int NQB);

// per-device state (device.cu): SM count of the current device; dynamic shared-memory opt-in of a
// kernel, set once per (device, kernel)
enum SmemKernel { kSmemFwdTcgen05 = 0, kSmemFwdTcgen05Log, kSmemSigTcgen05, kSmemScheduleItems, kSmemFwdMmaSync64,
                  kSmemFwdMmaSync128, kSmemMaskFromThreshold, kNumSmemKernels };
cudaError_t device_sm_count(int* n_sm);
cudaError_t ensure_dynamic_smem(SmemKernel id, const void* func, int bytes);

// launchers (each returns the cudaError_t of its launches; *n_launch += kernels enqueued)
cudaError_t launch_schedule(const FwdParams& p, const FwdWorkspace& w, int rows_per_item,
                            cudaStream_t st, int* n_launch, bool reuse = false);
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
cudaError_t launch_enumerate(const uint32_t* mask_bits, int H, int NQB, int NKB, int32_t* idx,
                             int32_t* cnt, cudaStream_t st);

}  // namespace sa

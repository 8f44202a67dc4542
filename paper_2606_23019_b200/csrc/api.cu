// api.cu -- the C ABI of libscalingattn.so (include/scalingattn.h): argument validation, error
// reporting, workspace carving and kernel dispatch. No arithmetic of the method lives here.
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "common.cuh"

namespace {

thread_local char g_err[512] = "";
thread_local int g_last_launches = 0;
std::atomic<int> g_variant{0};   // debug hook (sa_set_fwd_variant): read once per call

sa_status fail(sa_status s, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return s;
}

sa_status cuda_fail(cudaError_t e, const char* what) {
  return fail(SA_ERR_CUDA, "%s: %s (%s)", what, cudaGetErrorString(e), cudaGetErrorName(e));
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

constexpr int kMaxBlocksPerRow = 12288;  // shared-memory bound of the schedule pre-pass
constexpr int kMaxGroups = 8192;         // B*H bound of the schedule pre-pass

// compute capability of the current device must be 10.x (sm_100a binary)
sa_status check_device() {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
  static std::mutex mu;
  static int cached_dev = -1, cached_major = 0;
  std::lock_guard<std::mutex> lk(mu);
  if (cached_dev != dev) {
    int major = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaDeviceGetAttribute");
    cached_dev = dev;
    cached_major = major;
  }
  if (cached_major != 10)
    return fail(SA_ERR_UNSUPPORTED, "device compute capability %d.x; this library is sm_100a only",
                cached_major);
  return SA_OK;
}

sa_status validate_shape(int B, int H, int N, int n_valid, int D, int Bq, int Bk, float scale) {
  if (B <= 0 || H <= 0 || N <= 0 || D <= 0 || Bq <= 0 || Bk <= 0)
    return fail(SA_ERR_INVALID_ARG, "sizes must be positive (B=%d H=%d N=%d D=%d Bq=%d Bk=%d)", B,
                H, N, D, Bq, Bk);
  if (!((D == 128 && Bq == 128 && Bk == 128) || (D == 64 && Bq == 64 && Bk == 64)))
    return fail(SA_ERR_UNSUPPORTED,
                "(D,Bq,Bk)=(%d,%d,%d) unsupported; supported: (128,128,128), (64,64,64)", D, Bq, Bk);
  if (N % Bq != 0 || N % Bk != 0)
    return fail(SA_ERR_INVALID_ARG, "N=%d must be a multiple of Bq=%d and Bk=%d", N, Bq, Bk);
  if (n_valid < 1 || n_valid > N)
    return fail(SA_ERR_INVALID_ARG, "n_valid=%d outside [1, N=%d]", n_valid, N);
  if (!(scale > 0.f) || !(scale < 3.0e38f))
    return fail(SA_ERR_INVALID_ARG, "scale must be finite and positive");
  if (N / Bq > kMaxBlocksPerRow || static_cast<long long>(B) * H > kMaxGroups)
    return fail(SA_ERR_UNSUPPORTED, "N/Bq=%d > %d or B*H=%lld > %d", N / Bq, kMaxBlocksPerRow,
                static_cast<long long>(B) * H, kMaxGroups);
  return SA_OK;
}

// optional device timing of the dominant kernel (sa_profile_enable / sa_profile_collect)
std::mutex g_prof_mu;
std::vector<cudaEvent_t> g_prof_ev;   // 2 * capacity events: start, stop per forward call
int g_prof_n = 0;                     // forward calls recorded since the last collect

void prof_free() {
  for (cudaEvent_t e : g_prof_ev) cudaEventDestroy(e);
  g_prof_ev.clear();
  g_prof_n = 0;
}

// Internal workspaces of the short-signature call, one per (device, stream): the workspace holds the
// scheduler cursor and the work list, which a call rebuilds while an earlier call's persistent kernel
// may still be consuming them -- safe only in stream order. Calls on the same stream are ordered by
// the stream (the mutex is held across the enqueue, so two threads sharing a stream cannot interleave
// their launches); calls on different streams get different buffers. Buffers are allocated and, when
// they have to grow, freed in stream order (cudaMallocAsync / cudaFreeAsync on the caller's stream),
// so a buffer is never released while work that uses it is pending.
struct StreamWs {
  int dev;
  cudaStream_t stream;
  void* ptr;
  size_t bytes;
};
std::mutex g_ws_mu;
std::vector<StreamWs> g_ws;

// Copy engines for the host-buffer entry points: the q/k/v upload of head group g+1 and the out/lse
// download of group g-1 overlap the forward pass of group g (PCIe is full duplex and the copy engines
// run beside the SMs). Two non-blocking streams and a pool of events, created on first use.
struct PipeCtx {
  cudaStream_t h2d = nullptr, d2h = nullptr;
  std::vector<cudaEvent_t> ev;
  cudaError_t init(size_t n_events) {
    cudaError_t e = cudaSuccess;
    if (!h2d && (e = cudaStreamCreateWithFlags(&h2d, cudaStreamNonBlocking)) != cudaSuccess) return e;
    if (!d2h && (e = cudaStreamCreateWithFlags(&d2h, cudaStreamNonBlocking)) != cudaSuccess) return e;
    while (ev.size() < n_events) {
      cudaEvent_t x;
      if ((e = cudaEventCreateWithFlags(&x, cudaEventDisableTiming)) != cudaSuccess) return e;
      ev.push_back(x);
    }
    return e;
  }
};
std::mutex g_pipe_mu;
constexpr int kMaxPipeDevices = 64;
PipeCtx g_pipes[kMaxPipeDevices];   // streams and events belong to a device: one context per ordinal
constexpr int kPipeGroups = 8;     // head groups per batch entry (fewer when H is small)
// First head of group g (g = groups: H). The groups taper towards the end -- weights 3 3 3 3 3 3 2 1 -- so
// that what cannot overlap anything, the last group's compute and download, is short.
static int pipe_group_begin(int H, int groups, int g) {
  if (groups < kPipeGroups) return static_cast<int>(static_cast<long long>(H) * g / groups);   // one head each
  static const int cum[kPipeGroups + 1] = {0, 3, 6, 9, 12, 15, 18, 20, 21};
  int prev = 0;
  for (int i = 1; i <= g; ++i) {
    int h = static_cast<int>((static_cast<long long>(H) * cum[i] * 2 + 21) / 42);   // round(H cum / 21)
    h = h < prev + 1 ? prev + 1 : h;                                                 // every group has a head
    const int room = H - (groups - i);                                               // and leaves one for each later group
    prev = h > room ? room : h;
  }
  return prev;
}

}  // namespace

extern "C" {

int sa_mask_words_per_row(int N, int Bk) {
  if (N <= 0 || Bk <= 0 || N % Bk != 0) return -1;
  return (N / Bk + 31) / 32;
}

size_t sa_pack_mask_workspace_bytes(int H, int NQB, int NKB) {
  if (H <= 0 || NQB <= 0 || NKB <= 0) return 0;
  return sa::pack_mask_workspace_bytes(H, NQB, NKB);
}

// The workspace holds room for the parts of the last round's rows (sa::fwd_tail_plan), which depends
// on the SM count of the current device (148 when no device can be queried: sizing only).
static sa::TailPlan sized_tail_plan(int B, int H, int NQB) {
  int n_sm = 0;
  if (sa::device_sm_count(&n_sm) != cudaSuccess || n_sm <= 0) {
    (void)cudaGetLastError();
    n_sm = 148;
  }
  return sa::fwd_tail_plan(B, H, NQB, NQB < 0xFFFF ? NQB : 0xFFFF, n_sm);   // (the fast path has Bq == Bk)
}

size_t sa_fwd_workspace_bytes(int B, int H, int N, int Bq) {
  if (B <= 0 || H <= 0 || N <= 0 || Bq <= 0 || N % Bq != 0) return 0;
  return sa::fwd_workspace_bytes(B, H, N / Bq, (N / Bq + 31) / 32, sized_tail_plan(B, H, N / Bq));   // (Bq == Bk where parts exist)
}

static size_t al256(size_t x) { return (x + 255) / 256 * 256; }

// The host forms run the forward pass head group by head group (kPipeGroups chunks per batch entry,
// pipelined with the copies), every chunk through the same workspace: the largest chunk call's need
// (a chunk's plan for its last round differs from the whole problem's).
static size_t host_pipeline_ws_bytes(int H, int N, int Bq) {
  const int groups = H < kPipeGroups ? H : kPipeGroups;
  size_t need = 0;
  for (int g = 0; g < groups; ++g) {
    const int h0 = pipe_group_begin(H, groups, g), h1 = pipe_group_begin(H, groups, g + 1);
    const size_t n = sa_fwd_workspace_bytes(1, h1 - h0, N, Bq);
    need = n > need ? n : need;
  }
  return need;
}

size_t sa_fwd_host_scratch_bytes(int B, int H, int N, int D, int Bq, int Bk) {
  if (B <= 0 || H <= 0 || N <= 0 || D <= 0 || Bq <= 0 || Bk <= 0 || N % Bq || N % Bk) return 0;
  const size_t t = al256(static_cast<size_t>(B) * H * N * D * 2);
  const size_t l = al256(static_cast<size_t>(B) * H * N * 4);
  const size_t m = al256(static_cast<size_t>(H) * (N / Bq) * ((N / Bk + 31) / 32) * 4);
  return 4 * t + l + m + host_pipeline_ws_bytes(H, N, Bq);
}

sa_status sa_pack_mask(const float* scores, const float* density, uint32_t* mask_bits, int H,
                       int NQB, int NKB, int force_diag, void* workspace, size_t workspace_bytes,
                       void* stream) {
  if (!scores || !density || !mask_bits)
    return fail(SA_ERR_INVALID_ARG, "sa_pack_mask: null pointer");
  if (H <= 0 || NQB <= 0 || NKB <= 0)
    return fail(SA_ERR_INVALID_ARG, "sa_pack_mask: sizes must be positive (H=%d NQB=%d NKB=%d)", H,
                NQB, NKB);
  if (static_cast<long long>(NQB) * NKB > 0x7FFFFFFFLL)
    return fail(SA_ERR_UNSUPPORTED, "sa_pack_mask: NQB*NKB exceeds 2^31-1");
  if (!aligned16(scores) || !aligned16(mask_bits) || !aligned16(workspace))
    return fail(SA_ERR_INVALID_ARG, "sa_pack_mask: pointers must be 16-byte aligned");
  const size_t need = sa::pack_mask_workspace_bytes(H, NQB, NKB);
  if (!workspace || workspace_bytes < need)
    return fail(SA_ERR_WORKSPACE, "sa_pack_mask: workspace %zu B < %zu B", workspace_bytes, need);
  sa_status s = check_device();
  if (s != SA_OK) return s;
  cudaError_t e = sa::launch_pack_mask(scores, density, mask_bits, H, NQB, NKB, force_diag ? 1 : 0,
                                       workspace, static_cast<cudaStream_t>(stream));
  if (e != cudaSuccess) return cuda_fail(e, "sa_pack_mask launch");
  g_last_launches = sa::kPackMaskLaunches;
  return SA_OK;
}

sa_status sa_pack_mask_static(const float* scores, const float* density, uint32_t* mask_bits, int H,
                              int NQB, int NKB, int force_diag, void* stream) {
  g_last_launches = 0;
  if (!scores || !density || !mask_bits)
    return fail(SA_ERR_INVALID_ARG, "sa_pack_mask_static: null pointer");
  if (H <= 0 || NQB <= 0 || NKB <= 0)
    return fail(SA_ERR_INVALID_ARG, "sa_pack_mask_static: sizes must be positive (H=%d NQB=%d NKB=%d)", H,
                NQB, NKB);
  if (static_cast<long long>(NQB) * NKB > 0x7FFFFFFFLL)
    return fail(SA_ERR_UNSUPPORTED, "sa_pack_mask_static: NQB*NKB exceeds 2^31-1");
  if (!aligned16(scores) || !aligned16(mask_bits))
    return fail(SA_ERR_INVALID_ARG, "sa_pack_mask_static: pointers must be 16-byte aligned");
  const size_t need = sa::pack_mask_workspace_bytes(H, NQB, NKB);
  if (need > static_cast<size_t>(SA_STATIC_SCRATCH_BYTES))
    return fail(SA_ERR_WORKSPACE,
                "sa_pack_mask_static: H=%d NQB=%d NKB=%d needs %zu B of scratch, the library's fixed array "
                "holds %zu B (use sa_pack_mask with a workspace of your own)",
                H, NQB, NKB, need, static_cast<size_t>(SA_STATIC_SCRATCH_BYTES));
  sa_status s = check_device();
  if (s != SA_OK) return s;
  void* scratch = nullptr;
  size_t scratch_bytes = 0;
  cudaError_t e = sa::static_scratch(&scratch, &scratch_bytes);      // device address, looked up once per device
  if (e != cudaSuccess) return cuda_fail(e, "sa_pack_mask_static: cudaGetSymbolAddress(static scratch)");
  e = sa::launch_pack_mask(scores, density, mask_bits, H, NQB, NKB, force_diag ? 1 : 0, scratch,
                           static_cast<cudaStream_t>(stream));
  if (e != cudaSuccess) return cuda_fail(e, "sa_pack_mask_static launch");
  g_last_launches = sa::kPackMaskLaunches;
  return SA_OK;
}

sa_status sa_mask_from_threshold(const float* tmap, const float* p_star, uint32_t* mask_bits, int H,
                                 int nbq, int nbk, int NQB, int NKB, int force_diag, void* stream) {
  g_last_launches = 0;
  if (!tmap || !p_star || !mask_bits)
    return fail(SA_ERR_INVALID_ARG, "sa_mask_from_threshold: null pointer");
  if (H <= 0 || nbq <= 0 || nbk <= 0 || NQB <= 0 || NKB <= 0)
    return fail(SA_ERR_INVALID_ARG,
                "sa_mask_from_threshold: sizes must be positive (H=%d nbq=%d nbk=%d NQB=%d NKB=%d)", H,
                nbq, nbk, NQB, NKB);
  if (!aligned16(tmap) || !aligned16(mask_bits))
    return fail(SA_ERR_INVALID_ARG, "sa_mask_from_threshold: pointers must be 16-byte aligned");
  if (H > 65535 || nbq > 32768 || nbk > 32768 || NQB > 32768 || NKB > 32768 ||
      static_cast<long long>(H) * NQB * ((NKB + 31) / 32) > 0x3FFFFFFFLL)
    return fail(SA_ERR_UNSUPPORTED,
                "sa_mask_from_threshold: H > 65535, a grid side exceeds 32768 blocks or the mask 2^30 words");
  sa_status s = check_device();
  if (s != SA_OK) return s;
  cudaError_t e = sa::launch_mask_from_threshold(tmap, p_star, mask_bits, H, nbq, nbk, NQB, NKB,
                                                 force_diag ? 1 : 0,
                                                 static_cast<cudaStream_t>(stream));
  if (e != cudaSuccess) return cuda_fail(e, "sa_mask_from_threshold launch");
  g_last_launches = 1;
  return SA_OK;
}

sa_status sa_block_significance(const void* q, const void* k, const float* lse, float* sig, int B,
                                int H, int N, int n_valid, int D, int Bq, int Bk, float scale,
                                void* stream) {
  g_last_launches = 0;
  if (!q || !k || !lse || !sig) return fail(SA_ERR_INVALID_ARG, "sa_block_significance: null pointer");
  sa_status s = validate_shape(B, H, N, n_valid, D, Bq, Bk, scale);
  if (s != SA_OK) return s;
  if (D != 128) return fail(SA_ERR_UNSUPPORTED, "sa_block_significance: only (D,Bq,Bk) = (128,128,128)");
  if (!aligned16(q) || !aligned16(k))
    return fail(SA_ERR_INVALID_ARG, "sa_block_significance: q, k must be 16-byte aligned");
  s = check_device();
  if (s != SA_OK) return s;
  const char* txt = nullptr;
  cudaError_t e = sa::launch_block_significance(static_cast<const __nv_bfloat16*>(q),
                                                static_cast<const __nv_bfloat16*>(k), lse, sig, B, H, N,
                                                n_valid, scale, static_cast<cudaStream_t>(stream), &txt);
  if (e != cudaSuccess) return cuda_fail(e, txt ? txt : "sa_block_significance launch");
  g_last_launches = 1;
  return SA_OK;
}

size_t sa_threshold_map_update_workspace_bytes(int B, int H, int NQB, int NKB) {
  if (B <= 0 || H <= 0 || NQB <= 0 || NKB <= 0) return 0;
  if (static_cast<long long>(B) * H * NQB * NKB > 0x7FFFFFFFLL) return 0;
  return sa::threshold_update_workspace_bytes(B, H, NQB, NKB);
}

sa_status sa_threshold_map_update(const float* sig, const float* levels, int n_levels, float* tmap, int B,
                                  int H, int NQB, int NKB, void* workspace, size_t workspace_bytes,
                                  void* stream) {
  g_last_launches = 0;
  if (!sig || !levels || !tmap) return fail(SA_ERR_INVALID_ARG, "sa_threshold_map_update: null pointer");
  if (B <= 0 || H <= 0 || NQB <= 0 || NKB <= 0 || n_levels <= 0)
    return fail(SA_ERR_INVALID_ARG, "sa_threshold_map_update: sizes must be positive");
  if (n_levels > sa::kMaxThresholdLevels || static_cast<long long>(B) * H * NQB * NKB > 0x7FFFFFFFLL)
    return fail(SA_ERR_UNSUPPORTED, "sa_threshold_map_update: n_levels > %d or B*H*NQB*NKB >= 2^31",
                sa::kMaxThresholdLevels);
  const size_t need = sa::threshold_update_workspace_bytes(B, H, NQB, NKB);
  if (!workspace || workspace_bytes < need || (reinterpret_cast<uintptr_t>(workspace) & 255u))
    return fail(SA_ERR_WORKSPACE, "sa_threshold_map_update: workspace %zu B < %zu B or not 256 B aligned",
                workspace_bytes, need);
  sa_status s = check_device();
  if (s != SA_OK) return s;
  cudaError_t e = sa::launch_threshold_update(sig, levels, n_levels, tmap, B, H, NQB, NKB, workspace,
                                              static_cast<cudaStream_t>(stream), &g_last_launches);
  if (e != cudaSuccess) return cuda_fail(e, "sa_threshold_map_update launch");
  return SA_OK;
}

sa_status sa_fidelity_from_lse(const float* lse_dense, const float* lse_sparse, const int32_t* rows,
                               int n_rows, int B, int H, int N, float* fidelity, float* per_row,
                               void* stream) {
  g_last_launches = 0;
  if (!lse_dense || !lse_sparse || !rows || !fidelity)
    return fail(SA_ERR_INVALID_ARG, "sa_fidelity_from_lse: null pointer");
  if (n_rows <= 0 || B <= 0 || H <= 0 || N <= 0)
    return fail(SA_ERR_INVALID_ARG, "sa_fidelity_from_lse: sizes must be positive (n_rows=%d B=%d H=%d N=%d)",
                n_rows, B, H, N);
  if (static_cast<long long>(B) * H > 0x7FFFFFFFLL)
    return fail(SA_ERR_UNSUPPORTED, "sa_fidelity_from_lse: B*H exceeds 2^31-1");
  sa_status s = check_device();
  if (s != SA_OK) return s;
  cudaError_t e = sa::launch_fidelity(lse_dense, lse_sparse, rows, n_rows, B * H, N, fidelity, per_row,
                                      static_cast<cudaStream_t>(stream));
  if (e != cudaSuccess) return cuda_fail(e, "sa_fidelity_from_lse launch");
  g_last_launches = 1;
  return SA_OK;
}

// mask_word_aligned: the pipelined host entry points pass the mask of a head GROUP, which starts at a
// word boundary inside the caller's 16-byte aligned mask (the kernels read the mask word by word).
static sa_status fwd_ex_impl(const void* q, const void* k, const void* v, const uint32_t* mask_bits,
                             void* out, float* lse, int B, int H, int N, int n_valid, int D, int Bq,
                             int Bk, float scale, void* workspace, size_t workspace_bytes, void* stream,
                             bool mask_word_aligned, bool reuse_schedule = false,
                             int32_t* walk_log = nullptr) {
  g_last_launches = 0;
  if (!q || !k || !v || !mask_bits || !out || !lse)
    return fail(SA_ERR_INVALID_ARG, "sa_block_sparse_attn_fwd: null pointer");
  sa_status s = validate_shape(B, H, N, n_valid, D, Bq, Bk, scale);
  if (s != SA_OK) return s;
  const bool mask_ok = mask_word_aligned ? (reinterpret_cast<uintptr_t>(mask_bits) & 3u) == 0
                                        : aligned16(mask_bits);
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(out) || !mask_ok ||
      !aligned16(lse) || !aligned16(workspace))
    return fail(SA_ERR_INVALID_ARG, "sa_block_sparse_attn_fwd: pointers must be 16-byte aligned");
  const sa::TailPlan sized_plan = sized_tail_plan(B, H, N / Bq);
  const size_t need = sa::fwd_workspace_bytes(B, H, N / Bq, (N / Bq + 31) / 32, sized_plan);
  if (!workspace || workspace_bytes < need)
    return fail(SA_ERR_WORKSPACE, "sa_block_sparse_attn_fwd: workspace %zu B < %zu B",
                workspace_bytes, need);
  s = check_device();
  if (s != SA_OK) return s;

  cudaStream_t st = static_cast<cudaStream_t>(stream);
  sa::FwdParams p;
  p.q = static_cast<const __nv_bfloat16*>(q);
  p.k = static_cast<const __nv_bfloat16*>(k);
  p.v = static_cast<const __nv_bfloat16*>(v);
  p.mask_bits = mask_bits;
  p.out = static_cast<__nv_bfloat16*>(out);
  p.lse = lse;
  p.B = B; p.H = H; p.N = N; p.n_valid = n_valid; p.D = D; p.Bq = Bq; p.Bk = Bk;
  p.NQB = N / Bq; p.NKB = N / Bk; p.W = (p.NKB + 31) / 32;
  p.scale = scale;
  p.scale_log2 = scale * 1.4426950408889634f;
  const sa::FwdWorkspace w = sa::carve_fwd_workspace(workspace, B, H, p.NQB, (p.NQB + 31) / 32, sized_plan);
  p.items = w.items;
  p.n_items_dev = w.n_items;
  p.counter = w.cursor;
  p.stats = w.stats;
  p.walk_log = walk_log;
  const int variant = walk_log ? 2 : g_variant.load(std::memory_order_relaxed);   // the walk log is the pair path's
  const bool fast = (variant != 1 && D == 128);
  // the per-row score bound saves ~6% of the attention kernel but costs one more (~8 us) launch:
  // not worth it on problems of a few thousand tiles, which then keep the exact running max
  const bool big = static_cast<long long>(B) * H * p.NQB * p.NKB >= 16384;
  p.kmax2 = (fast && (variant == 2 || (variant == 0 && big))) ? w.kmax2 : nullptr;
  // The tcgen05 kernel works on items of two tiles: a PAIR of query blocks that share their K/V tiles,
  // or ONE query block whose key blocks alternate between the two tiles (a split item, merged in the
  // epilogue; twice as many items of half the length). With P pairs on n SMs a launch takes about
  // ceil(P / n) pair items or ceil(2 P / n) split items of half the length per SM: split items are
  // taken when that rounding favours them and the problem is small (below two waves of pairs); from
  // there on the dynamic scheduler evens the rounding out and the shared K/V tiles of pairs win
  // (measured: N = 4096, H = 12 dense 150 -> 131 us with split items, N = 8192 dense 374 us with pairs
  // against 446 us).
  int n_sm = 0;
  cudaError_t e = sa::device_sm_count(&n_sm);
  if (e != cudaSuccess) return cuda_fail(e, "device query");
  const long long n_pairs = static_cast<long long>(B) * H * ((p.NQB + 1) / 2);
  const long long rounds_pairs = 2 * ((n_pairs + n_sm - 1) / n_sm), rounds_split = (2 * n_pairs + n_sm - 1) / n_sm;
  const bool small = n_pairs < 2LL * n_sm && rounds_split < rounds_pairs;
  const int rows_per_item = (fast && (variant == 2 || (variant == 0 && !small))) ? 2 : 1;
  p.rows_per_item = rows_per_item;
  p.split_rows = (fast && rows_per_item == 1) ? 1 : 0;
  // the partly filled last round of pair items is issued in parts over key ranges (schedule.cu)
  const sa::TailPlan plan = (fast && variant == 0 && rows_per_item == 2 && p.NKB <= 0xFFFF)
                                ? sa::fwd_tail_plan(B, H, p.NQB, p.NKB, n_sm) : sa::TailPlan{};
  // large problems without parts run the lean build of the kernel (no split items, no parts: the
  // one leftover row of an odd head becomes a single-row item there, which at >= 8 rounds is noise)
  p.lean_items = (fast && variant == 0 && rows_per_item == 2 && plan.parts == 0 && n_pairs >= 8LL * n_sm) ? 1 : 0;
  p.part_mask = w.part_mask;
  p.part_out = w.part_out;
  p.part_lse = w.part_lse;
  p.n_items = B * H * ((p.NQB + rows_per_item - 1) / rows_per_item) + plan.rem * (plan.parts - (plan.parts ? 1 : 0));
  e = sa::launch_schedule(p, w, rows_per_item, plan, st, &g_last_launches, reuse_schedule);
  if (e != cudaSuccess) return cuda_fail(e, "schedule pre-pass launch");
  cudaEvent_t ev_stop = nullptr;
  {
    std::lock_guard<std::mutex> lk(g_prof_mu);
    if (2 * static_cast<size_t>(g_prof_n) + 1 < g_prof_ev.size()) {
      e = cudaEventRecord(g_prof_ev[2 * g_prof_n], st);
      if (e != cudaSuccess) return cuda_fail(e, "cudaEventRecord(profile start)");
      ev_stop = g_prof_ev[2 * g_prof_n + 1];
      ++g_prof_n;
    }
  }
  if (fast) {
    const char* txt = nullptr;
    e = sa::launch_fwd_tcgen05(p, nullptr, st, &g_last_launches, &txt);
    if (e != cudaSuccess) return cuda_fail(e, txt ? txt : "tcgen05 forward launch");
    e = sa::launch_combine_parts(p, w, plan, st, &g_last_launches);
    if (e != cudaSuccess) return cuda_fail(e, "combine launch");
  } else {
    e = sa::launch_fwd_mma_sync(p, st, &g_last_launches);
    if (e != cudaSuccess) return cuda_fail(e, "mma.sync forward launch");
  }
  if (ev_stop) {
    e = cudaEventRecord(ev_stop, st);
    if (e != cudaSuccess) return cuda_fail(e, "cudaEventRecord(profile stop)");
  }
  return SA_OK;
}

sa_status sa_block_sparse_attn_fwd_ex(const void* q, const void* k, const void* v,
                                      const uint32_t* mask_bits, void* out, float* lse, int B,
                                      int H, int N, int n_valid, int D, int Bq, int Bk,
                                      float scale, void* workspace, size_t workspace_bytes,
                                      void* stream) {
  return fwd_ex_impl(q, k, v, mask_bits, out, lse, B, H, N, n_valid, D, Bq, Bk, scale, workspace,
                     workspace_bytes, stream, false);
}

sa_status sa_debug_tail_plan(int B, int H, int N, int Bq, int Bk, int n_sm, int* rem, int* parts) {
  if (!rem || !parts || B <= 0 || H <= 0 || N <= 0 || Bq <= 0 || Bk <= 0 || N % Bq || N % Bk || n_sm <= 0)
    return fail(SA_ERR_INVALID_ARG, "sa_debug_tail_plan: bad sizes or null pointer");
  const sa::TailPlan t = sa::fwd_tail_plan(B, H, N / Bq, N / Bk, n_sm);
  *rem = t.rem;
  *parts = t.parts;
  return SA_OK;
}

size_t sa_debug_fwd_walk_log_bytes(int B, int H, int N, int Bq, int Bk) {
  if (B <= 0 || H <= 0 || N <= 0 || Bq <= 0 || Bk <= 0 || N % Bq || N % Bk) return 0;
  const size_t rows = static_cast<size_t>(B) * H * (N / Bq), nkb = static_cast<size_t>(N / Bk);
  return (3 * rows + 3 * rows * nkb) * sizeof(int32_t);
}

sa_status sa_debug_fwd_walk(const void* q, const void* k, const void* v, const uint32_t* mask_bits,
                            void* out, float* lse, int B, int H, int N, int n_valid, int D, int Bq,
                            int Bk, float scale, void* workspace, size_t workspace_bytes,
                            int32_t* walk_log, size_t walk_log_bytes, void* stream) {
  if (D != 128 || Bq != 128 || Bk != 128)
    return fail(SA_ERR_UNSUPPORTED, "sa_debug_fwd_walk: only (D,Bq,Bk) = (128,128,128)");
  const size_t need = sa_debug_fwd_walk_log_bytes(B, H, N, Bq, Bk);
  if (!walk_log || need == 0 || walk_log_bytes < need)
    return fail(SA_ERR_WORKSPACE, "sa_debug_fwd_walk: walk_log %zu B < %zu B", walk_log_bytes, need);
  return fwd_ex_impl(q, k, v, mask_bits, out, lse, B, H, N, n_valid, D, Bq, Bk, scale, workspace,
                     workspace_bytes, stream, false, false, walk_log);
}

sa_status sa_block_sparse_attn_fwd_reuse(const void* q, const void* k, const void* v,
                                         const uint32_t* mask_bits, void* out, float* lse, int B,
                                         int H, int N, int n_valid, int D, int Bq, int Bk,
                                         float scale, void* workspace, size_t workspace_bytes,
                                         void* stream) {
  return fwd_ex_impl(q, k, v, mask_bits, out, lse, B, H, N, n_valid, D, Bq, Bk, scale, workspace,
                     workspace_bytes, stream, false, true);
}

sa_status sa_block_sparse_attn_fwd(const void* q, const void* k, const void* v,
                                   const uint32_t* mask_bits, void* out, float* lse, int B, int H,
                                   int N, int D, int Bq, int Bk, float scale, void* stream) {
  const size_t need = sa_fwd_workspace_bytes(B, H, N, Bq);
  if (need == 0) return fail(SA_ERR_INVALID_ARG, "sa_block_sparse_attn_fwd: bad sizes");
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  std::lock_guard<std::mutex> lk(g_ws_mu);          // held until the call's kernels are enqueued
  StreamWs* slot = nullptr;
  for (StreamWs& w : g_ws)
    if (w.dev == dev && w.stream == st) slot = &w;
  if (!slot) {
    g_ws.push_back(StreamWs{dev, st, nullptr, 0});
    slot = &g_ws.back();
  }
  if (slot->bytes < need) {
    if (slot->ptr) {
      e = cudaFreeAsync(slot->ptr, st);             // after the stream's pending work that uses it
      if (e != cudaSuccess) return cuda_fail(e, "cudaFreeAsync(internal workspace)");
      slot->ptr = nullptr;
      slot->bytes = 0;
    }
    e = cudaMallocAsync(&slot->ptr, need, st);
    if (e != cudaSuccess) return cuda_fail(e, "cudaMallocAsync(internal workspace)");
    slot->bytes = need;
  }
  return sa_block_sparse_attn_fwd_ex(q, k, v, mask_bits, out, lse, B, H, N, N, D, Bq, Bk, scale,
                                     slot->ptr, need, stream);
}

// q, k, v up / forward / out, lse down, pipelined over head groups (see PipeCtx). The mask is already
// on the device. Everything is ordered after the work queued on `st` so far, and `st` waits for the
// last download, so callers see plain stream semantics.
static sa_status pipelined_fwd_host(const void* q_host, const void* k_host, const void* v_host,
                                    void* out_host, float* lse_host, char* dq, char* dk, char* dv,
                                    char* dout, char* dlse, const char* dmask, char* dws, int B, int H,
                                    int N, int n_valid, int D, int Bq, int Bk, float scale,
                                    cudaStream_t st, int* launches) {
  const int groups = H < kPipeGroups ? H : kPipeGroups;
  const int n_chunks = B * groups;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= kMaxPipeDevices)
    return cuda_fail(e != cudaSuccess ? e : cudaErrorInvalidDevice, "cudaGetDevice");
  std::lock_guard<std::mutex> lk(g_pipe_mu);
  PipeCtx& g_pipe = g_pipes[dev];
  e = g_pipe.init(2 * static_cast<size_t>(n_chunks) + 2);
  if (e != cudaSuccess) return cuda_fail(e, "copy pipeline setup");
  cudaEvent_t ev_start = g_pipe.ev[0], ev_end = g_pipe.ev[1];
  if ((e = cudaEventRecord(ev_start, st)) != cudaSuccess ||
      (e = cudaStreamWaitEvent(g_pipe.h2d, ev_start, 0)) != cudaSuccess ||
      (e = cudaStreamWaitEvent(g_pipe.d2h, ev_start, 0)) != cudaSuccess)
    return cuda_fail(e, "copy pipeline fork");
  const size_t row_bytes = static_cast<size_t>(N) * D * 2;
  const size_t mask_head_bytes = static_cast<size_t>(N / Bq) * ((N / Bk + 31) / 32) * 4;
  const size_t ws_bytes = host_pipeline_ws_bytes(H, N, Bq);
  int c = 0;
  for (int b = 0; b < B; ++b) {
    for (int g = 0; g < groups; ++g, ++c) {
      const int h0 = pipe_group_begin(H, groups, g), h1 = pipe_group_begin(H, groups, g + 1);
      const size_t off = (static_cast<size_t>(b) * H + h0) * row_bytes;
      const size_t bytes = static_cast<size_t>(h1 - h0) * row_bytes;
      const size_t loff = (static_cast<size_t>(b) * H + h0) * N * 4, lbytes = static_cast<size_t>(h1 - h0) * N * 4;
      cudaEvent_t ev_in = g_pipe.ev[2 + 2 * c], ev_done = g_pipe.ev[3 + 2 * c];
      if ((e = cudaMemcpyAsync(dq + off, static_cast<const char*>(q_host) + off, bytes, cudaMemcpyHostToDevice, g_pipe.h2d)) != cudaSuccess ||
          (e = cudaMemcpyAsync(dk + off, static_cast<const char*>(k_host) + off, bytes, cudaMemcpyHostToDevice, g_pipe.h2d)) != cudaSuccess ||
          (e = cudaMemcpyAsync(dv + off, static_cast<const char*>(v_host) + off, bytes, cudaMemcpyHostToDevice, g_pipe.h2d)) != cudaSuccess ||
          (e = cudaEventRecord(ev_in, g_pipe.h2d)) != cudaSuccess ||
          (e = cudaStreamWaitEvent(st, ev_in, 0)) != cudaSuccess)
        return cuda_fail(e, "host->device copy (q, k, v)");
      sa_status s = fwd_ex_impl(
          dq + off, dk + off, dv + off,
          reinterpret_cast<const uint32_t*>(dmask + static_cast<size_t>(h0) * mask_head_bytes), dout + off,
          reinterpret_cast<float*>(dlse + loff), 1, h1 - h0, N, n_valid, D, Bq, Bk, scale, dws, ws_bytes,
          st, true);
      if (s != SA_OK) return s;
      *launches += g_last_launches;
      if ((e = cudaEventRecord(ev_done, st)) != cudaSuccess ||
          (e = cudaStreamWaitEvent(g_pipe.d2h, ev_done, 0)) != cudaSuccess ||
          (e = cudaMemcpyAsync(static_cast<char*>(out_host) + off, dout + off, bytes, cudaMemcpyDeviceToHost, g_pipe.d2h)) != cudaSuccess ||
          (e = cudaMemcpyAsync(reinterpret_cast<char*>(lse_host) + loff, dlse + loff, lbytes, cudaMemcpyDeviceToHost, g_pipe.d2h)) != cudaSuccess)
        return cuda_fail(e, "device->host copy");
    }
  }
  if ((e = cudaEventRecord(ev_end, g_pipe.d2h)) != cudaSuccess ||
      (e = cudaStreamWaitEvent(st, ev_end, 0)) != cudaSuccess)
    return cuda_fail(e, "copy pipeline join");
  return SA_OK;
}

sa_status sa_block_sparse_attn_fwd_host(const void* q_host, const void* k_host, const void* v_host,
                                        const uint32_t* mask_bits_host, void* out_host,
                                        float* lse_host, int B, int H, int N, int n_valid, int D,
                                        int Bq, int Bk, float scale, void* scratch,
                                        size_t scratch_bytes, void* stream) {
  if (!q_host || !k_host || !v_host || !mask_bits_host || !out_host || !lse_host)
    return fail(SA_ERR_INVALID_ARG, "sa_block_sparse_attn_fwd_host: null pointer");
  sa_status s = validate_shape(B, H, N, n_valid, D, Bq, Bk, scale);
  if (s != SA_OK) return s;
  const size_t need = sa_fwd_host_scratch_bytes(B, H, N, D, Bq, Bk);
  if (!scratch || scratch_bytes < need || (reinterpret_cast<uintptr_t>(scratch) & 255u))
    return fail(SA_ERR_WORKSPACE, "sa_block_sparse_attn_fwd_host: scratch %zu B < %zu B or not 256 B aligned",
                scratch_bytes, need);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const size_t tb = static_cast<size_t>(B) * H * N * D * 2, t = al256(tb);
  const size_t lb = static_cast<size_t>(B) * H * N * 4, l = al256(lb);
  const size_t mb = static_cast<size_t>(H) * (N / Bq) * ((N / Bk + 31) / 32) * 4, m = al256(mb);
  char* base = static_cast<char*>(scratch);
  char *dq = base, *dk = base + t, *dv = base + 2 * t, *dout = base + 3 * t;
  char* dlse = base + 4 * t;
  char* dmask = dlse + l;
  char* dws = dmask + m;
  cudaError_t e;
  if ((e = cudaMemcpyAsync(dmask, mask_bits_host, mb, cudaMemcpyHostToDevice, st)) != cudaSuccess)
    return cuda_fail(e, "host->device copy (mask)");
  int launches = 0;
  s = pipelined_fwd_host(q_host, k_host, v_host, out_host, lse_host, dq, dk, dv, dout, dlse, dmask, dws, B,
                         H, N, n_valid, D, Bq, Bk, scale, st, &launches);
  if (s != SA_OK) return s;
  g_last_launches = launches;
  return SA_OK;
}

size_t sa_hot_path_host_scratch_bytes(int B, int H, int N, int D, int Bq, int Bk) {
  const size_t f = sa_fwd_host_scratch_bytes(B, H, N, D, Bq, Bk);
  if (f == 0) return 0;
  const int NQB = N / Bq, NKB = N / Bk;
  return f + al256(static_cast<size_t>(H) * NQB * NKB * 4) + al256(static_cast<size_t>(H) * 4) +
         al256(sa_pack_mask_workspace_bytes(H, NQB, NKB));
}

sa_status sa_hot_path_host(const float* scores_host, const float* density_host, int force_diag,
                           const void* q_host, const void* k_host, const void* v_host,
                           uint32_t* mask_bits_host, void* out_host, float* lse_host, int B, int H,
                           int N, int n_valid, int D, int Bq, int Bk, float scale, void* scratch,
                           size_t scratch_bytes, void* stream) {
  if (!scores_host || !density_host || !q_host || !k_host || !v_host || !mask_bits_host ||
      !out_host || !lse_host)
    return fail(SA_ERR_INVALID_ARG, "sa_hot_path_host: null pointer");
  sa_status s = validate_shape(B, H, N, n_valid, D, Bq, Bk, scale);
  if (s != SA_OK) return s;
  const size_t need = sa_hot_path_host_scratch_bytes(B, H, N, D, Bq, Bk);
  if (!scratch || scratch_bytes < need || (reinterpret_cast<uintptr_t>(scratch) & 255u))
    return fail(SA_ERR_WORKSPACE, "sa_hot_path_host: scratch %zu B < %zu B or not 256 B aligned",
                scratch_bytes, need);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int NQB = N / Bq, NKB = N / Bk;
  const size_t tb = static_cast<size_t>(B) * H * N * D * 2, t = al256(tb);
  const size_t lb = static_cast<size_t>(B) * H * N * 4, l = al256(lb);
  const size_t mb = static_cast<size_t>(H) * NQB * ((NKB + 31) / 32) * 4, m = al256(mb);
  const size_t sb = static_cast<size_t>(H) * NQB * NKB * 4, db = static_cast<size_t>(H) * 4;
  const size_t fwd_ws = host_pipeline_ws_bytes(H, N, Bq);
  const size_t pack_ws = sa_pack_mask_workspace_bytes(H, NQB, NKB);
  char* base = static_cast<char*>(scratch);
  char *dq = base, *dk = base + t, *dv = base + 2 * t, *dout = base + 3 * t;
  char* dlse = base + 4 * t;
  char* dmask = dlse + l;
  char* dws = dmask + m;
  char* dscores = dws + fwd_ws;            // fwd_ws is a multiple of 256
  char* ddens = dscores + al256(sb);
  char* dpws = ddens + al256(db);
  cudaError_t e;
  if ((e = cudaMemcpyAsync(dscores, scores_host, sb, cudaMemcpyHostToDevice, st)) != cudaSuccess ||
      (e = cudaMemcpyAsync(ddens, density_host, db, cudaMemcpyHostToDevice, st)) != cudaSuccess)
    return cuda_fail(e, "host->device copy (scores)");
  s = sa_pack_mask(reinterpret_cast<const float*>(dscores), reinterpret_cast<const float*>(ddens),
                   reinterpret_cast<uint32_t*>(dmask), H, NQB, NKB, force_diag, dpws, pack_ws,
                   stream);
  if (s != SA_OK) return s;
  int launches = sa::kPackMaskLaunches;
  s = pipelined_fwd_host(q_host, k_host, v_host, out_host, lse_host, dq, dk, dv, dout, dlse, dmask, dws, B,
                         H, N, n_valid, D, Bq, Bk, scale, st, &launches);
  if (s != SA_OK) return s;
  g_last_launches = launches;
  if ((e = cudaMemcpyAsync(mask_bits_host, dmask, mb, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
    return cuda_fail(e, "device->host copy (mask)");
  return SA_OK;
}

sa_status sa_profile_enable(int capacity) {
  std::lock_guard<std::mutex> lk(g_prof_mu);
  prof_free();
  if (capacity < 0) return fail(SA_ERR_INVALID_ARG, "sa_profile_enable: capacity %d < 0", capacity);
  for (int i = 0; i < 2 * capacity; ++i) {
    cudaEvent_t ev;
    cudaError_t e = cudaEventCreate(&ev);
    if (e != cudaSuccess) {
      prof_free();
      return cuda_fail(e, "cudaEventCreate");
    }
    g_prof_ev.push_back(ev);
  }
  return SA_OK;
}

sa_status sa_profile_collect(float* ms_host, int capacity, int* count_host) {
  if (!ms_host || !count_host || capacity < 0)
    return fail(SA_ERR_INVALID_ARG, "sa_profile_collect: bad arguments");
  std::lock_guard<std::mutex> lk(g_prof_mu);
  const int n = g_prof_n < capacity ? g_prof_n : capacity;
  for (int i = 0; i < n; ++i) {
    cudaError_t e = cudaEventSynchronize(g_prof_ev[2 * i + 1]);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms_host[i], g_prof_ev[2 * i], g_prof_ev[2 * i + 1]);
    if (e != cudaSuccess) return cuda_fail(e, "sa_profile_collect");
  }
  *count_host = n;
  g_prof_n = 0;
  return SA_OK;
}

sa_status sa_enumerate_active_blocks(const uint32_t* mask_bits, int H, int NQB, int NKB,
                                     int32_t* idx, int32_t* cnt, void* stream) {
  if (!mask_bits || !idx || !cnt)
    return fail(SA_ERR_INVALID_ARG, "sa_enumerate_active_blocks: null pointer");
  if (H <= 0 || NQB <= 0 || NKB <= 0)
    return fail(SA_ERR_INVALID_ARG, "sa_enumerate_active_blocks: sizes must be positive");
  sa_status s = check_device();
  if (s != SA_OK) return s;
  cudaError_t e = sa::launch_enumerate(mask_bits, H, NQB, NKB, idx, cnt,
                                       static_cast<cudaStream_t>(stream));
  if (e != cudaSuccess) return cuda_fail(e, "sa_enumerate_active_blocks launch");
  return SA_OK;
}

sa_status sa_fwd_softmax_path_counts(const void* workspace, long long* fixed_host, long long* exact_host,
                                     void* stream) {
  if (!workspace || !fixed_host || !exact_host)
    return fail(SA_ERR_INVALID_ARG, "sa_fwd_softmax_path_counts: null pointer");
  int32_t c[2] = {0, 0};
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  cudaError_t e = cudaMemcpyAsync(c, static_cast<const int32_t*>(workspace) + 2, sizeof c,
                                  cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return cuda_fail(e, "sa_fwd_softmax_path_counts");
  *fixed_host = c[0];
  *exact_host = c[1];
  return SA_OK;
}

sa_status sa_debug_ex2_rate(int iters, float* sink, float* ms_host, double* n_exp_host, void* stream) {
  if (!sink || !ms_host || !n_exp_host || iters <= 0)
    return fail(SA_ERR_INVALID_ARG, "sa_debug_ex2_rate: bad arguments");
  sa_status s = check_device();
  if (s != SA_OK) return s;
  int n_sm = 0;
  cudaError_t e = sa::device_sm_count(&n_sm);
  if (e != cudaSuccess) return cuda_fail(e, "device query");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  cudaEvent_t a = nullptr, b = nullptr;
  if ((e = cudaEventCreate(&a)) != cudaSuccess || (e = cudaEventCreate(&b)) != cudaSuccess) {
    if (a) cudaEventDestroy(a);
    return cuda_fail(e, "cudaEventCreate");
  }
  e = cudaEventRecord(a, st);
  if (e == cudaSuccess) e = sa::launch_ex2_rate(iters, sink, n_sm, st, n_exp_host);
  if (e == cudaSuccess) e = cudaEventRecord(b, st);
  if (e == cudaSuccess) e = cudaEventSynchronize(b);
  if (e == cudaSuccess) e = cudaEventElapsedTime(ms_host, a, b);
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  if (e != cudaSuccess) return cuda_fail(e, "sa_debug_ex2_rate");
  return SA_OK;
}

sa_status sa_debug_l2_fill_rate(const void* buf, size_t buf_bytes, int iters, float* ms_host,
                                double* bytes_host, void* stream) {
  if (!buf || !ms_host || !bytes_host || iters <= 0 || buf_bytes < 32768 || !aligned16(buf))
    return fail(SA_ERR_INVALID_ARG, "sa_debug_l2_fill_rate: bad arguments");
  sa_status s = check_device();
  if (s != SA_OK) return s;
  int n_sm = 0;
  cudaError_t e = sa::device_sm_count(&n_sm);
  if (e != cudaSuccess) return cuda_fail(e, "device query");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  cudaEvent_t a = nullptr, b = nullptr;
  if ((e = cudaEventCreate(&a)) != cudaSuccess || (e = cudaEventCreate(&b)) != cudaSuccess) {
    if (a) cudaEventDestroy(a);
    return cuda_fail(e, "cudaEventCreate");
  }
  e = cudaEventRecord(a, st);
  if (e == cudaSuccess) e = sa::launch_l2_fill(buf, buf_bytes, iters, n_sm, st, bytes_host);
  if (e == cudaSuccess) e = cudaEventRecord(b, st);
  if (e == cudaSuccess) e = cudaEventSynchronize(b);
  if (e == cudaSuccess) e = cudaEventElapsedTime(ms_host, a, b);
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  if (e != cudaSuccess) return cuda_fail(e, "sa_debug_l2_fill_rate");
  return SA_OK;
}

sa_status sa_set_fwd_variant(int variant) {
  if (variant < 0 || variant > 3)
    return fail(SA_ERR_INVALID_ARG, "sa_set_fwd_variant: variant %d not in {0,1,2,3}", variant);
  g_variant.store(variant, std::memory_order_relaxed);
  return SA_OK;
}
int sa_get_fwd_variant(void) { return g_variant.load(std::memory_order_relaxed); }
int sa_last_launch_count(void) { return g_last_launches; }

const char* sa_status_string(sa_status s) {
  switch (s) {
    case SA_OK: return "SA_OK";
    case SA_ERR_INVALID_ARG: return "SA_ERR_INVALID_ARG";
    case SA_ERR_UNSUPPORTED: return "SA_ERR_UNSUPPORTED";
    case SA_ERR_CUDA: return "SA_ERR_CUDA";
    case SA_ERR_WORKSPACE: return "SA_ERR_WORKSPACE";
  }
  return "SA_ERR_UNKNOWN";
}
const char* sa_last_error(void) { return g_err; }

}  // extern "C"

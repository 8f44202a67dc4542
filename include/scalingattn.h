/* scalingattn.h -- C ABI of libscalingattn.so: the B200 (sm_100a) hot path of ScalingAttention,
 * the bit-wise block-sparse attention forward pass the paper calls the "crm kernel".
 *
 * Citations are line numbers of the paper text /root/reference/PAPER.md.
 *
 * Conventions (all entry points):
 *  - Pointers are DEVICE pointers unless the parameter name ends in _host. The caller owns every
 *    buffer; the library never frees or retains a caller pointer past the stream-ordered end of
 *    the call, and never allocates device memory (scratch comes in as `workspace`; the short
 *    sa_block_sparse_attn_fwd keeps one lazily grown internal workspace per (device, stream) instead).
 *  - `stream` is a cudaStream_t passed as void*. Calls enqueue work on it and return without
 *    synchronising; outputs are valid once the stream reaches the end of the enqueued work.
 *  - Errors are return codes; nothing is launched when validation fails; sa_last_error() holds a
 *    thread-local detail string for the last non-OK status. No exceptions, no abort.
 *  - Results are deterministic: each (batch, head, query block) is reduced by one CTA over its
 *    active key blocks in ascending order; no atomics touch out or lse.
 *  - Supported shapes: (D, Bq, Bk) in {(128,128,128), (64,64,64)}. Anything else is
 *    SA_ERR_UNSUPPORTED, never a silent slow path. The device must be compute capability 10.x.
 *
 * Compressed Row Mask (CRM) layout (Sec. 4.3.2; bit order from Alg. 2,
 * INDEX = base + CTZ(val), base += 32 per word):
 *    mask_bits: uint32 [H][NQB][W], NQB = N/Bq, NKB = N/Bk, W = ceil(NKB/32);
 *    key block v of query block u of head h is active  <=>  bit (v % 32) of word (v / 32) of row
 *    (h, u) is 1. Bits at positions >= NKB are ignored by the forward pass and written as 0 by
 *    sa_pack_mask. The mask is per head and shared across the batch.
 */
#ifndef SCALINGATTN_H_
#define SCALINGATTN_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define SA_API __attribute__((visibility("default")))
#else
#define SA_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  SA_OK = 0,
  SA_ERR_INVALID_ARG = 1, /* null pointer, non-positive size, N % Bq/Bk != 0, n_valid outside [1,N],
                             misaligned pointer (16 B), bad variant id */
  SA_ERR_UNSUPPORTED = 2, /* (D,Bq,Bk) outside the supported set, or not an sm_100 device */
  SA_ERR_CUDA = 3,        /* a CUDA runtime / driver call failed; text in sa_last_error() */
  SA_ERR_WORKSPACE = 4    /* workspace null or smaller than the *_workspace_bytes() figure */
} sa_status;

/* Words per CRM bit-row = ceil((N/Bk)/32) (256k tokens, 128-blocks -> 64 words).
 * Host helper, no CUDA call. Returns -1 for non-positive arguments or N % Bk != 0. */
SA_API int sa_mask_words_per_row(int N, int Bk);

/* Bytes of device scratch the calls below need. Host helpers, no CUDA call; 0 on bad arguments. */
SA_API size_t sa_pack_mask_workspace_bytes(int H, int NQB, int NKB);
SA_API size_t sa_fwd_workspace_bytes(int B, int H, int N, int Bq);
/* Device staging a sa_block_sparse_attn_fwd_host call needs (q,k,v,out,lse,mask + fwd workspace). */
SA_API size_t sa_fwd_host_scratch_bytes(int B, int H, int N, int D, int Bq, int Bk);

/* Mask instantiation (PAPER.md:103 M_p = 1(T <= p); Alg. 1 l.31 PAPER.md:437) in the form
 * "per-head top-fraction of block scores -> packed bits" (readings P1-P4):
 *   scores  : fp32 [H][NQB][NKB] row-major, finite (NaN sorts lowest; -0 == +0)
 *   density : fp32 [H]; head h keeps k_h = clamp(floor((double)density[h]*NQB*NKB + 0.5), 1, NQB*NKB)
 *             blocks, taken in (score descending, flat index u*NKB+v ascending) order
 *   force_diag != 0: bits (u,u) are forced on, rank first and count towards k_h (k_h is raised
 *             to min(NQB,NKB) if smaller)
 *   mask_bits (out): uint32 [H][NQB][W]; exactly k_h bits set per head.
 * Bit-exact and deterministic. workspace >= sa_pack_mask_workspace_bytes(H,NQB,NKB), 16 B aligned. */
SA_API sa_status sa_pack_mask(const float* scores, const float* density, uint32_t* mask_bits, int H,
                       int NQB, int NKB, int force_diag, void* workspace, size_t workspace_bytes,
                       void* stream);

/* sa_pack_mask for callers that cannot allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): same operation, same arguments and results, but
 * the workspace is a fixed array inside the library, SA_STATIC_SCRATCH_BYTES (2.25 MiB) of device
 * memory that every GPU which loads the library holds until the process exits. The call allocates
 * and frees nothing (no cudaMalloc / cudaFree, no allocating library routine); the first call on a
 * device looks the array's address up (cudaGetSymbolAddress), later calls reuse it.
 * Limit: sa_pack_mask_workspace_bytes(H, NQB, NKB) <= SA_STATIC_SCRATCH_BYTES, e.g. H <= 64 heads at
 * up to 2048 x 2048 blocks; SA_ERR_WORKSPACE beyond it (the message names both sizes).
 * All calls on a device share the array: calls ordered on one stream (or by events) are safe, calls
 * that overlap on the GPU race on it and give undefined masks. Nothing is carried from call to call
 * (the histograms are zeroed on `stream` at the start of every call). Bit-exact and deterministic
 * like sa_pack_mask; 5 kernels and one memset on `stream`, no synchronisation. */
#define SA_STATIC_SCRATCH_BYTES (2304 * 1024)
SA_API sa_status sa_pack_mask_static(const float* scores, const float* density, uint32_t* mask_bits,
                                     int H, int NQB, int NKB, int force_diag, void* stream);

/* The paper's run-time mask path: a per-head THRESHOLD MAP kept at a base resolution, instantiated
 * at the target resolution (PAPER.md:103 M_p = 1(T <= p); Eq. 7, the conservative
 * bilinear resize with a ceiling rule; readings P14-P16):
 *   R_base[h][a][b]  = 1 if tmap[h][a][b] <= p_star[h] else 0              (fp32 comparison)
 *   bit (u,v) of head h = ceil( Phi(R_base[h], u*nbq/NQB, v*nbk/NKB) )     (Phi = bilinear, no
 *             half-cell offset, neighbours clamped to the last cell): on exactly when a base cell
 *             with positive interpolation weight is on. nbq == NQB and nbk == NKB gives 1(T <= p).
 *   force_diag != 0 additionally sets every bit (u,u).
 *   tmap    : fp32 [H][nbq][nbk] row-major (device);  p_star : fp32 [H] (device)
 *   mask_bits (out): uint32 [H][NQB][W], W = ceil(NKB/32), bits at positions >= NKB written 0.
 * Bit-exact and deterministic (integer index arithmetic only); one kernel on `stream`, no workspace,
 * no synchronisation. SA_ERR_INVALID_ARG for null / misaligned (16 B) pointers or non-positive sizes;
 * SA_ERR_UNSUPPORTED if a grid side exceeds 32768 blocks. */
SA_API sa_status sa_mask_from_threshold(const float* tmap, const float* p_star, uint32_t* mask_bits,
                                        int H, int nbq, int nbk, int NQB, int NKB, int force_diag,
                                        void* stream);

/* WEST's block-wise aggregation (Eq. 1; Alg. 1 l.9-10 PAPER.md:396-398) without
 * materialising the attention matrix: with lse the output of a forward call on the all-ones mask,
 *   sig[b][h][u][v] = (1/(Bq*Bk)) * sum_{i in block u, i < n_valid} sum_{j in block v, j < n_valid}
 *                     exp(scale * <q[b,h,i,:], k[b,h,j,:]> - lse[b,h,i])
 * (each valid query row spreads mass 1 over the key blocks; padded rows are left out, padded keys get
 * zero weight: DESIGN.md P18). A batch entry is one calibration sample.
 *   q, k : bf16 [B][H][N][D] (device, 16 B aligned);  lse : fp32 [B][H][N] (device)
 *   sig  : fp32 [B][H][N/Bq][N/Bk] (out, device)
 * Supported: (D,Bq,Bk) = (128,128,128) on sm_100 (SA_ERR_UNSUPPORTED otherwise). Deterministic. One
 * tcgen05 kernel on `stream`, no workspace, no synchronisation. */
SA_API sa_status sa_block_significance(const void* q, const void* k, const float* lse, float* sig,
                                       int B, int H, int N, int n_valid, int D, int Bq, int Bk,
                                       float scale, void* stream);

/* WEST's local threshold discovery and topology union (Alg. 1 l.12-17; DESIGN.md
 * readings P19-P20) for a batch of calibration samples. For every sample b and head h: sort the block
 * significances sig[b][h] in descending order (ties in flat-index order), C = inclusive cumulative sum
 * divided by its total; the blocks at sorted positions 0..tau(p) are active at level p, tau(p) the first
 * position with C >= p; L(u,v) = the smallest level at which (u,v) is active, 1.0 if none; then
 *   tmap[h][u][v] <- min(tmap[h][u][v], L(u,v))        (union over the samples of the batch).
 *   sig    : fp32 [B][H][NQB][NKB] (device), non-negative, e.g. from sa_block_significance
 *   levels : fp32 [n_levels] (device), ascending, in (0, 1], n_levels <= 256 (the candidate set P)
 *   tmap   : fp32 [H][NQB][NKB] (device, in/out); initialise with 1.0 before the first sample
 *   workspace >= sa_threshold_map_update_workspace_bytes(B,H,NQB,NKB) bytes, 256 B aligned.
 * The sort is the library's own stable radix sort (13 kernels in all); everything runs on `stream`
 * without synchronising. Deterministic. SA_ERR_UNSUPPORTED if B*H*NQB*NKB >= 2^31 or n_levels > 256. */
SA_API size_t sa_threshold_map_update_workspace_bytes(int B, int H, int NQB, int NKB);
SA_API sa_status sa_threshold_map_update(const float* sig, const float* levels, int n_levels, float* tmap,
                                         int B, int H, int NQB, int NKB, void* workspace,
                                         size_t workspace_bytes, void* stream);

/* FAST's Fidelity Score from the forward pass's log-sum-exp (Eq. 3 Hellinger distance,
 * PAPER.md:132-134 Eq. 4 F = 1 - H, PAPER.md:155-159 stratified row sample; reading P17):
 * with P the dense softmax row and P~ the softmax over the kept keys only,
 *   H(P, P~) = sqrt(1 - sqrt(rho)),  rho = exp(lse_sparse - lse_dense) = retained attention mass,
 * so for every (b,h):  fidelity[b][h] = mean over i < n_rows of 1 - H at query row rows[i].
 *   lse_dense, lse_sparse : fp32 [B][H][N] (device), the lse outputs of two forward calls on the same
 *                           q, k, scale, n_valid: all-ones mask and the candidate mask
 *   rows        : int32 [n_rows] (device), query-row indices in [0, N), drawn by the caller (e.g. a few
 *                 per row block, Sec. 4.2.3), shared by all (b,h); an index outside [0, N) makes the
 *                 affected outputs NaN
 *   fidelity    : fp32 [B][H] (out);   per_row : fp32 [B][H][n_rows] (out) or NULL
 * A row empty in both masks scores 1, a row whose kept set is empty scores 0. Deterministic. One kernel
 * on `stream`, no workspace, no synchronisation. */
SA_API sa_status sa_fidelity_from_lse(const float* lse_dense, const float* lse_sparse,
                                      const int32_t* rows, int n_rows, int B, int H, int N,
                                      float* fidelity, float* per_row, void* stream);

/* Block-sparse attention forward (Sec. 4.3.2; Alg. 2):
 *   out[b,h,i,:] = sum_j softmax_j(scale * <q[b,h,i,:], k[b,h,j,:]>) * v[b,h,j,:]
 *   lse[b,h,i]   = ln sum_j exp(scale * <q_i, k_j>)                       (natural log)
 * with j ranging over the tokens of the key blocks whose bit is set in row (h, i / Bq). Masked key
 * blocks are never loaded and never multiplied. A row with no active key gives out = 0, lse = -inf.
 *   q, k, v, out : bf16 [B][H][N][D] contiguous, 16 B aligned;  lse : fp32 [B][H][N]
 *   scale        : softmax scale (e.g. 1/sqrt(D)); arithmetic is bf16 x bf16 -> fp32.
 * All N tokens are real. Uses an internal workspace per (device, stream): the workspace holds the
 * scheduler cursor and the work list, which a call rebuilds while an earlier call's kernel may still
 * be consuming them, so sharing one is only safe in stream order. It is allocated on first use and
 * when a larger problem arrives, in stream order (cudaMallocAsync / cudaFreeAsync on `stream`, no
 * synchronisation), and kept until the process exits. Calls from several threads are serialised
 * across their enqueue (calls sharing a stream then run in the order the lock was taken). */
SA_API sa_status sa_block_sparse_attn_fwd(const void* q, const void* k, const void* v,
                                   const uint32_t* mask_bits, void* out, float* lse, int B, int H,
                                   int N, int D, int Bq, int Bk, float scale, void* stream);

/* Same, plus n_valid (keys >= n_valid get exactly zero weight, even inside an active block; query
 * rows >= n_valid are computed like any other row) and a caller-provided workspace of at least
 * sa_fwd_workspace_bytes(B,H,N,Bq) bytes (16 B aligned), so nothing is allocated in the call.
 * sa_fwd_workspace_bytes is for the CURRENT device: besides the work list the workspace holds the
 * partial results of the query blocks that a call issues in parts over key ranges (the partly filled
 * last round of work items over the device's SMs; merged by one more kernel of the same call), whose
 * number depends on the SM count. Deterministic: a given (shape, mask, SM count) always takes the same
 * parts, merged in a fixed order. 3 or 4 kernels on `stream`. */
SA_API sa_status sa_block_sparse_attn_fwd_ex(const void* q, const void* k, const void* v,
                                      const uint32_t* mask_bits, void* out, float* lse, int B,
                                      int H, int N, int n_valid, int D, int Bq, int Bk,
                                      float scale, void* workspace, size_t workspace_bytes,
                                      void* stream);

/* The static-mask form (Fig. 3(c) "Reuse for All Prompts"; masks are fixed
 * per layer, timestep and head and reused by every call): same as sa_block_sparse_attn_fwd_ex, but the
 * work list that an earlier _ex call left in `workspace` is reused instead of being rebuilt, so the
 * two schedule kernels are skipped (their ~14 us matter at short sequences). Precondition: `workspace`
 * was last filled by sa_block_sparse_attn_fwd_ex (or this call) on the same device with the same B, H,
 * N, Bq, Bk, the same forward variant and a mask with the same contents; the result is undefined
 * otherwise. */
SA_API sa_status sa_block_sparse_attn_fwd_reuse(const void* q, const void* k, const void* v,
                                         const uint32_t* mask_bits, void* out, float* lse, int B,
                                         int H, int N, int n_valid, int D, int Bq, int Bk,
                                         float scale, void* workspace, size_t workspace_bytes,
                                         void* stream);

/* End-to-end form with HOST buffers (pinned memory recommended): copies q, k, v and the mask to
 * `scratch` (device, >= sa_fwd_host_scratch_bytes, 256 B aligned), runs the forward pass there and
 * copies out and lse back, without synchronising. The work is ordered like work queued on `stream`
 * (it starts after what `stream` holds and `stream` waits for its end), but the uploads and downloads
 * run on two internal copy streams, pipelined over groups of heads, so that PCIe traffic in both
 * directions overlaps the forward pass. */
SA_API sa_status sa_block_sparse_attn_fwd_host(const void* q_host, const void* k_host, const void* v_host,
                                        const uint32_t* mask_bits_host, void* out_host,
                                        float* lse_host, int B, int H, int N, int n_valid, int D,
                                        int Bq, int Bk, float scale, void* scratch,
                                        size_t scratch_bytes, void* stream);

/* One pass of the whole hot path with HOST buffers (pinned memory recommended), all on `stream`,
 * without synchronising: copies scores [H][NQB][NKB] and density [H] to the device and packs the
 * mask (sa_pack_mask, force_diag as there), copies q, k, v, runs the forward pass, and copies out,
 * lse and the packed mask (mask_bits_host, uint32 [H][NQB][W], out) back; q, k, v / out, lse are
 * pipelined over head groups on internal copy streams as in sa_block_sparse_attn_fwd_host. `scratch` is device
 * memory of at least sa_hot_path_host_scratch_bytes(...) bytes, 256 B aligned. */
SA_API size_t sa_hot_path_host_scratch_bytes(int B, int H, int N, int D, int Bq, int Bk);
SA_API sa_status sa_hot_path_host(const float* scores_host, const float* density_host, int force_diag,
                           const void* q_host, const void* k_host, const void* v_host,
                           uint32_t* mask_bits_host, void* out_host, float* lse_host, int B, int H,
                           int N, int n_valid, int D, int Bq, int Bk, float scale, void* scratch,
                           size_t scratch_bytes, void* stream);

/* Device timing of the dominant kernel. sa_profile_enable(capacity > 0) creates `capacity` CUDA
 * event pairs; from then on each forward call records one pair on its stream around the
 * attention kernel alone (after the schedule pre-pass), until `capacity` calls have been recorded.
 * sa_profile_collect waits for the recorded pairs, writes their elapsed milliseconds to
 * ms_host[0..*count_host) (host memory, at most `capacity` entries) and starts over at pair 0.
 * sa_profile_enable(0) switches recording off and destroys the events. Process-wide; not for use
 * from several threads at once. */
SA_API sa_status sa_profile_enable(int capacity);
SA_API sa_status sa_profile_collect(float* ms_host, int capacity, int* count_host);

/* CRM forward iterator on the device (Alg. 2), exposed so that its walk can be
 * checked on its own: for every row (h,u) writes the active key blocks in the order the iterator
 * yields them to idx[h][u][0..cnt) (int32 [H][NQB][NKB]) and their number to cnt[h][u]
 * (int32 [H][NQB]). Entries of idx past cnt are left untouched. */
SA_API sa_status sa_enumerate_active_blocks(const uint32_t* mask_bits, int H, int NQB, int NKB,
                                     int32_t* idx, int32_t* cnt, void* stream);

/* Which CUDA kernel the forward pass uses. 0 (default): automatic -- the tcgen05/TMEM/TMA kernel
 * for (128,128,128), the mma.sync kernel for (64,64,64); the tcgen05 kernel takes work items of two
 * query blocks of one (batch, head) that share their K/V tiles (the schedule pre-pass pairs adjacent
 * blocks when their popcounts are balanced, otherwise blocks of similar popcount and large bit-row
 * overlap); on small problems (fewer than two waves of such pairs, when the rounding to whole items per
 * SM favours it) it takes single query blocks instead, each SPLIT over the kernel's two tiles (even key
 * blocks to one, odd to the other, merged in the epilogue). 1: the mma.sync kernel for every supported shape (a
 * second CUDA implementation kept for cross-checking; not a fallback: it is never chosen implicitly
 * for a shape the fast kernel supports). 2 / 3: the tcgen05 kernel with its large-problem path (pair
 * items, key-norm pre-pass and score bound) / its small-problem path (split single-block items, exact
 * running max) forced, so that tests can drive either on any size. A DEBUG hook for tests and benchmarks, not
 * part of the product surface: process-wide (an atomic read once per call), so it must not be changed
 * while another thread is inside a forward call. The same holds for sa_profile_enable / _collect. */
SA_API sa_status sa_set_fwd_variant(int variant);
SA_API int sa_get_fwd_variant(void);

/* Which softmax path the last forward call that used `workspace` took (tcgen05 kernel only; see
 * DESIGN.md K1): per (softmax warp, work item) with at least one key block, *fixed_host counts those
 * that fixed the reference point at the Cauchy-Schwarz score bound for the whole item and *exact_host
 * those that kept the exact running max (bound too loose for the row norms at hand, or no key-norm
 * pass on a small problem). Synchronises `stream`. Host pointers. */
SA_API sa_status sa_fwd_softmax_path_counts(const void* workspace, long long* fixed_host,
                                            long long* exact_host, void* stream);

/* Measurement hook for the roofline of sa_block_significance (bound: the special-function pipe):
 * runs one launch of a kernel in which every resident warp does nothing but independent
 * ex2.approx chains (`iters` rounds of 8 per thread) on `stream`, waits for it, and returns its
 * elapsed milliseconds in *ms_host and the number of exponentials it executed in *n_exp_host (host
 * pointers). `sink`: device memory, at least 8 * (number of SMs) floats, never written in practice.
 * Call it in a loop for a sustained-load figure. */
SA_API sa_status sa_debug_ex2_rate(int iters, float* sink, float* ms_host, double* n_exp_host, void* stream);

/* Measurement hook for the secondary bound of the attention kernel on masks whose work items share no
 * key blocks (every (query tile, key block) unit then needs 64 KB of K and V from L2): one CTA per SM
 * keeps six 32 KB bulk copies global -> shared memory in flight, `iters` copies per SM, walking `buf`
 * (device, 16 B aligned, `buf_bytes` >= 32 KB; a buffer that fits L2 is served from L2 after the first
 * pass). Runs one launch on `stream`, waits for it, returns its milliseconds in *ms_host and the bytes it
 * moved in *bytes_host (host pointers). */
SA_API sa_status sa_debug_l2_fill_rate(const void* buf, size_t buf_bytes, int iters, float* ms_host,
                                       double* bytes_host, void* stream);

/* Debug hook: sa_block_sparse_attn_fwd_ex on a build of the (128,128,128) tcgen05 kernel that also
 * records its walk, so that the union walk of a work item (Alg. 2 re-expressed over the OR of two
 * bit-rows), the numbering of (tile, key block) units and the 64-word window reload can be checked
 * index by index against a CPU enumeration. walk_log: device int32, sa_debug_fwd_walk_log_bytes(...)
 * bytes, zero-filled by the caller. With R = B*H*N/Bq rows (row = (b*H + h)*NQB + u) and NKB = N/Bk:
 *   wg_cnt [R]           units the softmax warpgroup of the row's tile consumed
 *   wg_info[R]           (partner + 1) << 1 | tile      (partner = the item's other query block, -1: none)
 *   wg_seq [R][NKB]      unit << 16 | key block, in consumption order (unit = number in the item's walk)
 *   is_cnt [R]           units the MMA issuer issued for the item whose tile 0 is this row
 *   is_seq [R][2*NKB]    tile << 15 | key block, in issue order
 * Results (out, lse) are those of the product kernel. Requires (D,Bq,Bk) = (128,128,128). */
SA_API size_t sa_debug_fwd_walk_log_bytes(int B, int H, int N, int Bq, int Bk);
SA_API sa_status sa_debug_fwd_walk(const void* q, const void* k, const void* v, const uint32_t* mask_bits,
                                   void* out, float* lse, int B, int H, int N, int n_valid, int D, int Bq,
                                   int Bk, float scale, void* workspace, size_t workspace_bytes,
                                   int32_t* walk_log, size_t walk_log_bytes, void* stream);

/* Debug hook (host arithmetic only, no CUDA call): the plan a forward call of this shape follows for the
 * partly filled last round of its pair items on a device with n_sm SMs (K2): *rem work
 * items (spread over the B*H groups, each group's lightest) are issued in *parts parts over key ranges
 * and merged afterwards; 0 / 0 when every item stays whole. SA_ERR_INVALID_ARG on bad sizes. */
SA_API sa_status sa_debug_tail_plan(int B, int H, int N, int Bq, int Bk, int n_sm, int* rem, int* parts);

/* Number of kernels the last sa_pack_mask / forward / sa_hot_path_host call on this thread
 * enqueued (for bench accounting; memsets and copies are not counted). */
SA_API int sa_last_launch_count(void);

SA_API const char* sa_status_string(sa_status s); /* static string, never freed */
SA_API const char* sa_last_error(void);           /* thread-local text for the last non-OK status */

#ifdef __cplusplus
}
#endif
#endif /* SCALINGATTN_H_ */

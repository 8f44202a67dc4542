// sa_oracle.cpp -- CPU ORACLE for the ScalingAttention hot path. TEST INFRASTRUCTURE ONLY.
//
// This file is the plain, slow, fp64 statement of what the CUDA path must compute. It is
// test infrastructure: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load it. It shares no code, header, table or helper with
// paper_2606_23019_b200/csrc (the product) and never includes anything from there.
//
// What it states (citations are /root/reference/PAPER.md line numbers):
//  * Compressed Row Mask (CRM) bit layout: "each attention row [is] a compact bitmask stored in
//    aligned uint32 arrays, where each bit indicates the activation of a KV block"
//    (Sec. 4.3.2). Alg. 2 returns INDEX = base + CTZ(val) with base advancing by
//    32 per word, which fixes the order: key block v <-> word v/32,
//    bit v%32 (LSB first). Here the bits are read with plain shifts, not with a bit-scan walk.
//  * Block-sparse attention: the crm kernel is FlashAttention with the dense KV-block iterator
//    replaced by the CRM iterator. FlashAttention's online softmax is an exact
//    reformulation of softmax attention, so the result has a plain definition: masked
//    softmax(scale * Q K^T) V restricted to the keys of active blocks. That definition is what
//    is written out below, token by token (readings P5-P8).
//  * Mask instantiation M = 1(T <= p*) (Sec. 4.1.2; Alg. 1 l.31 PAPER.md:437) in the
//    form BASELINE.json names: per-head top-fraction of block scores -> bits (P1-P4).
//
// Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): dense special case vs torch SDPA fp64,
// arbitrary mask vs SDPA with a token-level boolean mask, block-diagonal special case,
// weights sum to 1, long-double brute force without max subtraction, closed forms (V const,
// Q = 0), key-block permutation invariance, empty row, padding; pack: round trip, popcount,
// order statistics, torch.sort(stable) top-k, Alg. 2 iterator restated in the test, golden words.
// No function here is "parity unpinned".
//
// Build: g++ -O2 -std=c++17 -shared -fPIC -pthread (oracle/build.py). Not tuned; never will be.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <thread>
#include <vector>

namespace {

// bf16 bit pattern -> double, exactly (bf16 is the top 16 bits of an IEEE fp32).
inline double bf16_to_double(uint16_t bits) {
  uint32_t u = static_cast<uint32_t>(bits) << 16;
  float f;
  std::memcpy(&f, &u, sizeof f);
  return static_cast<double>(f);
}

inline int words_per_row(int nkb) { return (nkb + 31) / 32; }

// Bit (u, v) of head h. Plain shift-and-test (order from Alg. 2).
inline int mask_bit(const uint32_t* bits, int nqb, int nkb, int h, int u, int v) {
  const int W = words_per_row(nkb);
  const uint32_t word = bits[(static_cast<size_t>(h) * nqb + u) * W + v / 32];
  return static_cast<int>((word >> (v % 32)) & 1u);
}

template <class F>
void parallel_for(int n, int n_threads, F f) {
  if (n_threads <= 0) n_threads = static_cast<int>(std::thread::hardware_concurrency());
  if (n_threads < 1) n_threads = 1;
  if (n_threads > n) n_threads = n > 0 ? n : 1;
  if (n_threads == 1) {
    for (int i = 0; i < n; ++i) f(i);
    return;
  }
  std::vector<std::thread> pool;
  for (int t = 0; t < n_threads; ++t)
    pool.emplace_back([=]() {
      for (int i = t; i < n; i += n_threads) f(i);
    });
  for (auto& th : pool) th.join();
}

// One query token i of (b, h): the definition, O-1.
//   J = { j < n_valid : M[h][i / Bq][j / Bk] = 1 }
//   s_j = scale * <q_i, k_j>;  m = max s_j;  Z = sum exp(s_j - m)
//   w_j = exp(s_j - m) / Z;    out_i = sum_j w_j v_j;   lse_i = m + ln Z
// Empty J: out_i = 0, lse_i = -inf (P7). If `weights` is non-null it receives w (length
// N, zero outside J) so a test can check sum_j w_j = 1.
void attn_row(const uint16_t* q, const uint16_t* k, const uint16_t* v, const uint32_t* bits,
              int H, int N, int D, int Bq, int Bk, int n_valid, double scale, int b, int h, int i,
              double* out_row, double* lse_out, double* weights) {
  const int nqb = N / Bq, nkb = N / Bk;
  const size_t head_off = (static_cast<size_t>(b) * H + h) * static_cast<size_t>(N) * D;
  const uint16_t* qi = q + head_off + static_cast<size_t>(i) * D;
  const int u = i / Bq;

  std::vector<double> qd(D);
  for (int d = 0; d < D; ++d) qd[d] = bf16_to_double(qi[d]);

  std::vector<double> s(N, 0.0);
  std::vector<char> in_J(N, 0);
  bool any = false;
  double m = -std::numeric_limits<double>::infinity();
  for (int j = 0; j < n_valid; ++j) {
    if (!mask_bit(bits, nqb, nkb, h, u, j / Bk)) continue;
    const uint16_t* kj = k + head_off + static_cast<size_t>(j) * D;
    double dot = 0.0;
    for (int d = 0; d < D; ++d) dot += qd[d] * bf16_to_double(kj[d]);
    s[j] = scale * dot;
    in_J[j] = 1;
    any = true;
    if (s[j] > m) m = s[j];
  }
  for (int d = 0; d < D; ++d) out_row[d] = 0.0;
  if (weights) for (int j = 0; j < N; ++j) weights[j] = 0.0;
  if (!any) {
    *lse_out = -std::numeric_limits<double>::infinity();
    return;
  }
  double Z = 0.0;
  for (int j = 0; j < n_valid; ++j)
    if (in_J[j]) Z += std::exp(s[j] - m);
  for (int j = 0; j < n_valid; ++j) {
    if (!in_J[j]) continue;
    const double w = std::exp(s[j] - m) / Z;
    if (weights) weights[j] = w;
    const uint16_t* vj = v + head_off + static_cast<size_t>(j) * D;
    for (int d = 0; d < D; ++d) out_row[d] += w * bf16_to_double(vj[d]);
  }
  *lse_out = m + std::log(Z);
}

}  // namespace

extern "C" {

int oracle_hardware_threads(void) { return static_cast<int>(std::thread::hardware_concurrency()); }

int oracle_words_per_row(int N, int Bk) { return words_per_row(N / Bk); }

// bits uint32 [H][NQB][W] -> dense uint8 [H][NQB][NKB] (bit order PAPER.md:512,536).
void oracle_unpack_mask(const uint32_t* bits, uint8_t* dense, int H, int NQB, int NKB) {
  for (int h = 0; h < H; ++h)
    for (int u = 0; u < NQB; ++u)
      for (int v = 0; v < NKB; ++v)
        dense[(static_cast<size_t>(h) * NQB + u) * NKB + v] =
            static_cast<uint8_t>(mask_bit(bits, NQB, NKB, h, u, v));
}

// dense uint8 [H][NQB][NKB] -> bits uint32 [H][NQB][W]; bits at positions >= NKB are zero.
void oracle_pack_bool(const uint8_t* dense, uint32_t* bits, int H, int NQB, int NKB) {
  const int W = words_per_row(NKB);
  for (int h = 0; h < H; ++h)
    for (int u = 0; u < NQB; ++u) {
      uint32_t* row = bits + (static_cast<size_t>(h) * NQB + u) * W;
      for (int w = 0; w < W; ++w) row[w] = 0u;
      for (int v = 0; v < NKB; ++v)
        if (dense[(static_cast<size_t>(h) * NQB + u) * NKB + v]) row[v / 32] |= (1u << (v % 32));
    }
}

// Number of blocks head h keeps: round-half-up of density*total in fp64, clamped to [1,total],
// raised to the diagonal count when force_diag (P2, P3).
long long oracle_keep_count(float density, int NQB, int NKB, int force_diag) {
  const long long total = static_cast<long long>(NQB) * NKB;
  long long kh = static_cast<long long>(std::floor(static_cast<double>(density) * static_cast<double>(total) + 0.5));
  if (kh < 1) kh = 1;
  if (kh > total) kh = total;
  if (force_diag) {
    const long long ndiag = std::min(NQB, NKB);
    if (kh < ndiag) kh = ndiag;
  }
  return kh;
}

// Per-head top-fraction selection of block scores -> bits (O-2; Eq. 2 /
// M_p = 1(T <= p); density = fraction of active blocks).
//   order all (u,v) by (score descending, flat index ascending)  -> std::stable_sort
//   diagonal entries rank first when force_diag (key = +inf);  keep the first k_h.
// Returns 0, or 1 if a score is not finite (precondition, P4).
int oracle_pack_mask(const float* scores, const float* density, uint32_t* bits, int H, int NQB,
                     int NKB, int force_diag) {
  const int W = words_per_row(NKB);
  const size_t total = static_cast<size_t>(NQB) * NKB;
  for (int h = 0; h < H; ++h) {
    const float* sc = scores + static_cast<size_t>(h) * total;
    std::vector<double> key(total);
    for (size_t idx = 0; idx < total; ++idx) {
      if (!std::isfinite(sc[idx])) return 1;
      double x = static_cast<double>(sc[idx]);
      if (x == 0.0) x = 0.0;  // -0.0 and +0.0 compare equal already; stored as +0.0 for clarity
      key[idx] = x;
    }
    if (force_diag)
      for (int u = 0; u < std::min(NQB, NKB); ++u)
        key[static_cast<size_t>(u) * NKB + u] = std::numeric_limits<double>::infinity();
    std::vector<uint32_t> order(total);
    for (size_t idx = 0; idx < total; ++idx) order[idx] = static_cast<uint32_t>(idx);
    std::stable_sort(order.begin(), order.end(),
                     [&](uint32_t a, uint32_t b) { return key[a] > key[b]; });
    const long long kh = oracle_keep_count(density[h], NQB, NKB, force_diag);
    uint32_t* hb = bits + static_cast<size_t>(h) * NQB * W;
    for (size_t i = 0; i < static_cast<size_t>(NQB) * W; ++i) hb[i] = 0u;
    for (long long r = 0; r < kh; ++r) {
      const uint32_t idx = order[static_cast<size_t>(r)];
      const int u = static_cast<int>(idx / NKB), v = static_cast<int>(idx % NKB);
      hb[static_cast<size_t>(u) * W + v / 32] |= (1u << (v % 32));
    }
  }
  return 0;
}

// Full attention oracle: q,k,v bf16 bit patterns [B][H][N][D]; bits [H][NQB][W] shared across the
// batch (P10); out fp64 [B][H][N][D]; lse fp64 [B][H][N] (natural log, P6).
void oracle_attn(const uint16_t* q, const uint16_t* k, const uint16_t* v, const uint32_t* bits,
                 double* out, double* lse, int B, int H, int N, int D, int Bq, int Bk, int n_valid,
                 float scale, int n_threads) {
  const int rows = B * H * N;
  parallel_for(rows, n_threads, [=](int r) {
    const int i = r % N, h = (r / N) % H, b = r / (N * H);
    attn_row(q, k, v, bits, H, N, D, Bq, Bk, n_valid, static_cast<double>(scale), b, h, i,
             out + static_cast<size_t>(r) * D, lse + r, nullptr);
  });
}

// Same definition on a list of units (b, h, u) = units[3*t .. 3*t+2]: out fp64 [n_units][Bq][D],
// lse fp64 [n_units][Bq]. Used at the large configs where the full oracle is infeasible.
void oracle_attn_units(const uint16_t* q, const uint16_t* k, const uint16_t* v,
                       const uint32_t* bits, const int32_t* units, int n_units, double* out,
                       double* lse, int B, int H, int N, int D, int Bq, int Bk, int n_valid,
                       float scale, int n_threads) {
  (void)B;
  const int rows = n_units * Bq;
  parallel_for(rows, n_threads, [=](int r) {
    const int t = r / Bq, ii = r % Bq;
    const int b = units[3 * t], h = units[3 * t + 1], u = units[3 * t + 2];
    attn_row(q, k, v, bits, H, N, D, Bq, Bk, n_valid, static_cast<double>(scale), b, h,
             u * Bq + ii, out + static_cast<size_t>(r) * D, lse + r, nullptr);
  });
}

// Softmax weights of one query token (length N, zero outside the active valid keys), plus its
// output row and lse: lets a test check sum_j w_j = 1 and recompute out from w.
void oracle_attn_row_weights(const uint16_t* q, const uint16_t* k, const uint16_t* v,
                             const uint32_t* bits, int H, int N, int D, int Bq, int Bk,
                             int n_valid, float scale, int b, int h, int i, double* weights,
                             double* out_row, double* lse) {
  attn_row(q, k, v, bits, H, N, D, Bq, Bk, n_valid, static_cast<double>(scale), b, h, i, out_row,
           lse, weights);
}

}  // extern "C"

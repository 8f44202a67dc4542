// fidelity.cu -- sa_fidelity_from_lse: FAST's Fidelity Score from the log-sum-exp the forward pass
// already writes.
//
// Fidelity Score F(P, P~) = 1 - H(P, P~) (Eq. 4) with the Hellinger distance
// H(P,Q) = (1/sqrt 2) sqrt(sum_i (sqrt p_i - sqrt q_i)^2) (Eq. 3), averaged over
// a stratified sample of query rows (Sec. 4.2.3).
//
// With P the dense softmax row and P~ the softmax renormalised over the kept keys (DESIGN.md
// reading P17), sum_i sqrt(p_i q_i) = sqrt(rho), rho = Z~/Z the retained attention mass, so
//     H^2 = 1 - sqrt(rho),   rho = exp(lse_sparse - lse_dense):
// the whole N x N comparison collapses to one value per row that two forward calls (the dense mask
// and the candidate mask) have already produced. 1 - sqrt(rho) is evaluated as -expm1(d/2),
// d = lse_sparse - lse_dense <= 0, which keeps full precision when the mask drops little mass.
// One CTA per (b, h); fixed-order tree reduction (deterministic).
#include "common.cuh"

namespace sa {
namespace {

constexpr int kThreads = 256;

__global__ void __launch_bounds__(kThreads)
fidelity_kernel(const float* __restrict__ lse_dense, const float* __restrict__ lse_sparse,
                const int32_t* __restrict__ rows, int n_rows, int N, float* __restrict__ fidelity,
                float* __restrict__ per_row) {
  __shared__ float red[kThreads];
  const size_t base = static_cast<size_t>(blockIdx.x) * N;
  float acc = 0.f;
  for (int i = threadIdx.x; i < n_rows; i += kThreads) {
    const int r = __ldg(rows + i);
    const bool in_range = static_cast<unsigned>(r) < static_cast<unsigned>(N);
    const float ld = in_range ? __ldg(lse_dense + base + r) : 0.f;
    const float ls = in_range ? __ldg(lse_sparse + base + r) : 0.f;
    float f;
    if (!in_range) {
      f = __int_as_float(0x7FC00000);   // a row index outside [0, N) poisons the result with NaN
    } else if (ld == -INFINITY) {
      f = 1.f;                      // no key at all in either: identical (empty) rows
    } else if (ls == -INFINITY) {
      f = 0.f;                      // everything dropped: disjoint supports, H = 1
    } else {
      const float d = fminf(ls - ld, 0.f);                 // rounding can leave d a hair above 0
      f = 1.f - sqrtf(fmaxf(-expm1f(0.5f * d), 0.f));      // 1 - sqrt(1 - sqrt(rho))
    }
    if (per_row) per_row[static_cast<size_t>(blockIdx.x) * n_rows + i] = f;
    acc += f;
  }
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int s = kThreads / 2; s > 0; s >>= 1) {
    if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) fidelity[blockIdx.x] = red[0] / static_cast<float>(n_rows);
}

}  // namespace

cudaError_t launch_fidelity(const float* lse_dense, const float* lse_sparse, const int32_t* rows,
                            int n_rows, int BH, int N, float* fidelity, float* per_row,
                            cudaStream_t st) {
  fidelity_kernel<<<BH, kThreads, 0, st>>>(lse_dense, lse_sparse, rows, n_rows, N, fidelity, per_row);
  return cudaGetLastError();
}

}  // namespace sa

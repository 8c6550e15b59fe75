// lerf.cu — LERF-style relevancy score from the cosine map of legs_relevancy (optional;
// PAPER.md:360 "in accordance with LERF [18]"; the formula is not in the paper: DESIGN.md reading C-21b):
//   out[p][j] = min_i exp(tau c_pj) / (exp(tau c_pj) + exp(tau c_pi)),  j < n_pos <= i < Q.
// The pairwise softmax is decreasing in the negative's cosine, so the minimum over the negatives is taken at their
// maximum: out[p][j] = 1 / (1 + exp(tau (max_i c_pi - c_pj))). One thread per pixel, HBM-streaming (4 Q B in, 4 n_pos B out).
#include "common.cuh"

namespace {

constexpr int kLerfThreads = 256;

__global__ void __launch_bounds__(kLerfThreads) lerf_kernel(const float* __restrict__ cosines, long long P, int Q, int n_pos,
                                                            float tau, float* __restrict__ out) {
  const long long p = (long long)blockIdx.x * kLerfThreads + threadIdx.x;
  if (p >= P) return;
  const float* c = cosines + p * Q;
  float neg = -3.0e38f;
  for (int i = n_pos; i < Q; ++i) neg = fmaxf(neg, c[i]);
  for (int j = 0; j < n_pos; ++j) out[p * n_pos + j] = 1.0f / (1.0f + __expf(tau * (neg - c[j])));
}

}  // namespace

extern "C" int legs_relevancy_lerf(legs_ctx* ctx, const float* cosines, int64_t P, int32_t Q, int32_t n_pos, float tau,
                                   float* out, void* stream) {
  if (!ctx) return LEGS_ERR_NULL;
  if (P < 0 || Q < 2 || Q > 16 || n_pos < 1 || n_pos >= Q || !(tau >= 0.f) || !(tau <= 100.f)) return LEGS_ERR_DIM;
  if (P == 0) return LEGS_OK;
  if (!cosines || !out) return LEGS_ERR_NULL;
  if (!legs_aligned16(cosines) || !legs_aligned16(out)) return LEGS_ERR_ALIGN;
  lerf_kernel<<<(unsigned)((P + kLerfThreads - 1) / kLerfThreads), kLerfThreads, 0, (cudaStream_t)stream>>>(cosines, P, Q, n_pos,
                                                                                                        tau, out);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

// optim.cu — training-step plumbing named at PAPER.md:182: one fused multi-tensor Adam step
// ("Adam optimizer [25], with a learning rate set to 0.001 and betas equal to (0.9, 0.999)") over all attribute arrays of
// the Gaussians, and the per-view density-control statistics ("adaptive density control" following [17]) from the
// dmean2d that legs_render_backward produces. Both are HBM streaming kernels: 16 B read + 12 B written per parameter
// (p, g, m, v -> p, m, v); 12 B read + up to 12 B written per Gaussian.
#include "common.cuh"

namespace {

constexpr int kOptThreads = 256;
constexpr int kMaxTensors = 16;

struct AdamArgs {
  float* p[kMaxTensors];
  const float* g[kMaxTensors];
  float* m[kMaxTensors];
  float* v[kMaxTensors];
  long long end4[kMaxTensors];   // exclusive prefix end of each tensor, in float4 units (counts rounded up)
  long long count[kMaxTensors];  // floats
  int n;
  float lr_c1, b1, b2, eps, inv_sqrt_c2;   // lr / (1 - b1^t), betas, eps, 1 / sqrt(1 - b2^t)
};

__device__ __forceinline__ void adam_one(float& p, float g, float& m, float& v, const AdamArgs& a) {
  m = fmaf(a.b1, m, (1.0f - a.b1) * g);
  v = fmaf(a.b2, v, (1.0f - a.b2) * g * g);
  // p - lr (m / c1) / (sqrt(v / c2) + eps)
  p = p - (a.lr_c1 * m) / (sqrtf(v) * a.inv_sqrt_c2 + a.eps);
}

__global__ void __launch_bounds__(kOptThreads) adam_kernel(const __grid_constant__ AdamArgs a) {
  const long long total4 = a.end4[a.n - 1];
  for (long long i = (long long)blockIdx.x * kOptThreads + threadIdx.x; i < total4; i += (long long)gridDim.x * kOptThreads) {
    int t = 0;
    while (i >= a.end4[t]) ++t;
    const long long j4 = i - (t ? a.end4[t - 1] : 0), j = j4 * 4;
    float* p = a.p[t] + j;
    const float* g = a.g[t] + j;
    float* m = a.m[t] + j;
    float* v = a.v[t] + j;
    if (j + 4 <= a.count[t]) {
      float4 P = *reinterpret_cast<float4*>(p), M = *reinterpret_cast<float4*>(m), V = *reinterpret_cast<float4*>(v);
      const float4 G = *reinterpret_cast<const float4*>(g);
      adam_one(P.x, G.x, M.x, V.x, a); adam_one(P.y, G.y, M.y, V.y, a);
      adam_one(P.z, G.z, M.z, V.z, a); adam_one(P.w, G.w, M.w, V.w, a);
      *reinterpret_cast<float4*>(p) = P; *reinterpret_cast<float4*>(m) = M; *reinterpret_cast<float4*>(v) = V;
    } else {
      for (long long k = 0; j + k < a.count[t]; ++k) {
        float P = p[k], M = m[k], V = v[k];
        adam_one(P, g[k], M, V, a);
        p[k] = P; m[k] = M; v[k] = V;
      }
    }
  }
}

__global__ void __launch_bounds__(kOptThreads) density_stats_kernel(long long n, const float2* __restrict__ dmean2d,
                                                                    const int* __restrict__ radius,
                                                                    float* __restrict__ grad_accum,
                                                                    unsigned int* __restrict__ denom,
                                                                    int* __restrict__ max_radius) {
  const long long i = (long long)blockIdx.x * kOptThreads + threadIdx.x;
  if (i >= n) return;
  const int r = radius[i];
  if (r <= 0) return;
  const float2 d = dmean2d[i];
  grad_accum[i] += sqrtf(d.x * d.x + d.y * d.y);
  denom[i] += 1u;
  max_radius[i] = max(max_radius[i], r);
}

}  // namespace

extern "C" {

int legs_adam_step(legs_ctx* ctx, int32_t n_tensors, float* const* params, const float* const* grads, float* const* m,
                   float* const* v, const int64_t* counts, const legs_adam* hp, void* stream) {
  if (!ctx || !params || !grads || !m || !v || !counts || !hp) return LEGS_ERR_NULL;
  if (n_tensors < 1 || n_tensors > kMaxTensors || hp->step < 1) return LEGS_ERR_DIM;
  if (!(hp->beta1 >= 0.f && hp->beta1 < 1.f) || !(hp->beta2 >= 0.f && hp->beta2 < 1.f) || !(hp->eps >= 0.f)) return LEGS_ERR_DIM;
  AdamArgs a;
  long long run = 0;
  int k = 0;
  for (int t = 0; t < n_tensors; ++t) {
    if (counts[t] < 0) return LEGS_ERR_DIM;
    if (counts[t] == 0) continue;
    if (!params[t] || !grads[t] || !m[t] || !v[t]) return LEGS_ERR_NULL;
    if (!legs_aligned16(params[t]) || !legs_aligned16(grads[t]) || !legs_aligned16(m[t]) || !legs_aligned16(v[t]))
      return LEGS_ERR_ALIGN;
    a.p[k] = params[t]; a.g[k] = grads[t]; a.m[k] = m[t]; a.v[k] = v[t];
    a.count[k] = counts[t];
    run += (counts[t] + 3) / 4;
    a.end4[k] = run;
    ++k;
  }
  if (k == 0) return LEGS_OK;
  for (int t = k; t < kMaxTensors; ++t) { a.p[t] = nullptr; a.g[t] = nullptr; a.m[t] = nullptr; a.v[t] = nullptr; a.count[t] = 0; a.end4[t] = run; }
  a.n = k;
  // bias corrections in double on the host: 1 - b^t loses everything in fp32 for small t and b2 = 0.999
  const double c1 = 1.0 - pow((double)hp->beta1, (double)hp->step), c2 = 1.0 - pow((double)hp->beta2, (double)hp->step);
  a.lr_c1 = (float)((double)hp->lr / c1);
  a.inv_sqrt_c2 = (float)(1.0 / sqrt(c2));
  a.b1 = hp->beta1; a.b2 = hp->beta2; a.eps = hp->eps;
  const long long blocks = (run + kOptThreads - 1) / kOptThreads;
  const int grid = (int)(blocks < (long long)ctx->num_sms * 16 ? blocks : (long long)ctx->num_sms * 16);
  adam_kernel<<<grid, kOptThreads, 0, (cudaStream_t)stream>>>(a);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

int legs_density_stats(legs_ctx* ctx, int64_t n, const float* dmean2d, const int32_t* radius, float* grad_accum,
                       uint32_t* denom, int32_t* max_radius, void* stream) {
  if (!ctx) return LEGS_ERR_NULL;
  if (n < 0) return LEGS_ERR_DIM;
  if (n == 0) return LEGS_OK;
  if (!dmean2d || !radius || !grad_accum || !denom || !max_radius) return LEGS_ERR_NULL;
  if (!legs_aligned16(dmean2d) || !legs_aligned16(radius) || !legs_aligned16(grad_accum) || !legs_aligned16(denom) ||
      !legs_aligned16(max_radius))
    return LEGS_ERR_ALIGN;
  density_stats_kernel<<<(unsigned)((n + kOptThreads - 1) / kOptThreads), kOptThreads, 0, (cudaStream_t)stream>>>(
      n, (const float2*)dmean2d, radius, grad_accum, denom, max_radius);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

}  // extern "C"

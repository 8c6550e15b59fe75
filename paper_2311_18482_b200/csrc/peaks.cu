// peaks.cu — measurement kernels for the roofline denominators of the ALU-bound compositors ("measure
// it with an FMA-chain micro-benchmark in the same run"). Not part of the hot path: bench.py times
// these launches with CUDA events, clocks sampled, and divides the compositors' work by the measured rates.
//   kind 0: FFMA chains       -> FP32-pipe lane-instructions per second (one fma.rn.f32 = one lane-instruction)
//   kind 1: MUFU.EX2 chains   -> ex2.approx per second (the second ceiling of S5/S6/S9)
//   kind 2: packed fma.rn.f32x2 chains -> lane-instructions per second when two FP32 FMAs share one issue slot
//   kind 3: FFMA + SHFL mix (1 shuffle per 4 FMAs), the instruction mix of the backward reduction
#include "common.cuh"

namespace {

constexpr int kPeakThreads = 256;
constexpr int kChains = 8;   // independent dependency chains per thread (covers the 4-cycle FMA latency at 2+ warps/SMSP)

// m and c arrive as kernel arguments so that the FMAs are the 3-register form real code uses (the immediate form
// issues at twice the rate on this part and would overstate the peak).
template <int KIND>
__global__ void __launch_bounds__(kPeakThreads) peak_kernel(int iters, float seed, float m, float c,
                                                            float* __restrict__ sink) {
  float a[kChains];
#pragma unroll
  for (int k = 0; k < kChains; ++k) a[k] = seed + (float)(threadIdx.x + k) * 1e-3f;
  if (KIND == 0) {
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int k = 0; k < kChains; ++k) a[k] = fmaf(a[k], m, c);
    }
  } else if (KIND == 1) {
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int k = 0; k < kChains; ++k) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(a[k]));
    }
  } else if (KIND == 2) {
    unsigned long long p[kChains / 2], mm, cc;
    asm("mov.b64 %0, {%1, %1};" : "=l"(mm) : "f"(m));
    asm("mov.b64 %0, {%1, %1};" : "=l"(cc) : "f"(c));
#pragma unroll
    for (int k = 0; k < kChains / 2; ++k) asm("mov.b64 %0, {%1, %2};" : "=l"(p[k]) : "f"(a[2 * k]), "f"(a[2 * k + 1]));
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int k = 0; k < kChains / 2; ++k) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[k]) : "l"(mm), "l"(cc));
    }
#pragma unroll
    for (int k = 0; k < kChains / 2; ++k) asm("mov.b64 {%0, %1}, %2;" : "=f"(a[2 * k]), "=f"(a[2 * k + 1]) : "l"(p[k]));
  } else {
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int r = 0; r < 4; ++r) {
#pragma unroll
        for (int k = 0; k < kChains; ++k) a[k] = fmaf(a[k], m, c);
        a[r] += __shfl_xor_sync(0xffffffffu, a[r + 4], 1 << r);
        a[r + 4] += __shfl_xor_sync(0xffffffffu, a[r], 16 >> r);
      }
    }
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < kChains; ++k) s += a[k];
  if (s == 123.456f) sink[blockIdx.x * kPeakThreads + threadIdx.x] = s;   // never true: keeps the chains alive
}

}  // namespace

extern "C" int legs_peak_kernel(legs_ctx* ctx, int32_t kind, int32_t iters, float* sink, uint64_t* lane_ops_host,
                                void* stream) {
  if (!ctx || !sink || !lane_ops_host) return LEGS_ERR_NULL;
  if (kind < 0 || kind > 3 || iters <= 0) return LEGS_ERR_DIM;
  cudaStream_t st = (cudaStream_t)stream;
  const int grid = ctx->num_sms * 8;   // 8 CTAs x 8 warps per SM = 16 warps per SMSP
  switch (kind) {
    case 0: peak_kernel<0><<<grid, kPeakThreads, 0, st>>>(iters, 1.0f, 0.999f, 1e-3f, sink); break;
    case 1: peak_kernel<1><<<grid, kPeakThreads, 0, st>>>(iters, -1.0f, 0.999f, 1e-3f, sink); break;
    case 2: peak_kernel<2><<<grid, kPeakThreads, 0, st>>>(iters, 1.0f, 0.999f, 1e-3f, sink); break;
    default: peak_kernel<3><<<grid, kPeakThreads, 0, st>>>(iters, 1.0f, 0.999f, 1e-3f, sink); break;
  }
  LEGS_LAUNCH_CHECK(ctx);
  // counted operations per launch: FMA (or ex2) lane-operations; kind 2 counts two per packed instruction
  const uint64_t per_thread = (uint64_t)iters * 4 * kChains * (kind == 2 ? 2 : 1);
  *lane_ops_host = per_thread * (uint64_t)grid * kPeakThreads;
  return LEGS_OK;
}

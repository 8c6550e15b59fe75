// relevancy_map.cu — S11 from an already DECODED feature map (legs_relevancy's `input_is_probs = 0` case;
// PAPER.md:360 "the relevance map of F", read as the plain cosine of reading C-21):
//   rel[p][q] = <F_p[0:d_clip], query_q> / (|F_p[0:d_clip]| |query_q|),   F [P,d] bf16 (the `decoded` of legs_decode_semantics).
// For callers that hold only F (the probabilities were not kept). HBM-read-bound: 2 d_clip bytes per pixel (1 KB at
// d_clip = 512) against 8 d_clip Q flops, so the kernel is a stream over F; the dot products go through mma.sync
// (m16n8k16, bf16 x bf16 -> fp32) only to keep the instruction count per loaded byte independent of Q and well under the
// HBM time (a tcgen05 pipeline for an N = 8..16 contraction would spend its time on set-up; the tensor pipe is idle here
// either way). Each warp owns 16 pixel rows; a lane loads 16 contiguous bytes of row g (and of row g+8) per 32-column block.
// The mma k index is a permutation of the real column index, the same on the F side and on the query side (a dot product
// does not care): real columns 32 kb + 8 t + {0..3} feed k-step 0 (k = 2t, 2t+1, 2t+8, 2t+9), columns + {4..7} feed
// k-step 1, so one 16-byte load serves two k-steps on both operands. |F_p|^2 is accumulated in fp32 from the same registers.
#include "common.cuh"

namespace {

constexpr int kMapThreads = 256;   // 8 warps x 16 rows
constexpr int kMapQPad = 16;       // query rows in shared memory (two n = 8 tiles)
constexpr int kMapRowPad = 64;     // bytes: rows g and g+1 of the queries fall into different bank halves

__device__ __forceinline__ void mma_bf16_m16n8k16(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                                  uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

__device__ __forceinline__ float sumsq_bf16x8(uint4 v, float acc) {
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float lo = __uint_as_float(w[i] << 16), hi = __uint_as_float(w[i] & 0xffff0000u);
    acc = fmaf(lo, lo, acc);
    acc = fmaf(hi, hi, acc);
  }
  return acc;
}

template <int NT>   // NT = n tiles of 8 queries (1: Q <= 8, 2: Q <= 16)
__global__ void __launch_bounds__(kMapThreads) relevancy_map_kernel(const uint16_t* __restrict__ F, long long P, int d,
                                                                    int d_clip, const uint16_t* __restrict__ queries, int Q,
                                                                    float* __restrict__ rel) {
  extern __shared__ __align__(16) uint8_t smem[];
  const int kblocks = (d_clip + 31) / 32;
  const int pitch = kblocks * 64 + kMapRowPad;            // bytes per query row
  float* s_inv = reinterpret_cast<float*>(smem + kMapQPad * pitch);   // 1 / |query_q|
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // queries -> shared memory (bf16 as given, zero rows / columns beyond Q / d_clip), and their inverse norms
  for (int i = threadIdx.x; i < kMapQPad * (pitch / 16); i += kMapThreads) {
    const int q = i / (pitch / 16), ch = i % (pitch / 16);
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (q < Q && ch * 8 < d_clip) v = *reinterpret_cast<const uint4*>(queries + (size_t)q * d_clip + ch * 8);
    *reinterpret_cast<uint4*>(smem + q * pitch + ch * 16) = v;
  }
  __syncthreads();
  for (int q = warp; q < kMapQPad; q += kMapThreads / 32) {
    float acc = 0.f;
    for (int ch = lane; ch < kblocks * 4; ch += 32) acc = sumsq_bf16x8(*reinterpret_cast<const uint4*>(smem + q * pitch + ch * 16), acc);
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) s_inv[q] = acc > 0.f ? rsqrtf(acc) : 0.f;
  }
  __syncthreads();

  const int g = lane >> 2, t = lane & 3;
  const long long tiles = (P + 15) / 16;
  for (long long tile = (long long)blockIdx.x * (kMapThreads / 32) + warp; tile < tiles; tile += (long long)gridDim.x * (kMapThreads / 32)) {
    const long long r0 = tile * 16 + g, r1 = r0 + 8;
    const uint16_t* f0 = F + (size_t)(r0 < P ? r0 : 0) * d + 8 * t;
    const uint16_t* f1 = F + (size_t)(r1 < P ? r1 : 0) * d + 8 * t;
    float c[NT][4];
#pragma unroll
    for (int n = 0; n < NT; ++n) c[n][0] = c[n][1] = c[n][2] = c[n][3] = 0.f;
    float n0 = 0.f, n1 = 0.f;
#pragma unroll 4
    for (int kb = 0; kb < kblocks; ++kb) {
      const bool in = kb * 32 + 8 * t < d_clip;             // d_clip is a multiple of 8: a 16-byte chunk is in or out
      uint4 a = make_uint4(0u, 0u, 0u, 0u), b = a;
      if (in && r0 < P) a = __ldg(reinterpret_cast<const uint4*>(f0 + kb * 32));
      if (in && r1 < P) b = __ldg(reinterpret_cast<const uint4*>(f1 + kb * 32));
#pragma unroll
      for (int n = 0; n < NT; ++n) {
        const uint4 qv = *reinterpret_cast<const uint4*>(smem + (8 * n + g) * pitch + kb * 64 + 16 * t);
        mma_bf16_m16n8k16(c[n], a.x, b.x, a.y, b.y, qv.x, qv.y);
        mma_bf16_m16n8k16(c[n], a.z, b.z, a.w, b.w, qv.z, qv.w);
      }
      n0 = sumsq_bf16x8(a, n0);
      n1 = sumsq_bf16x8(b, n1);
    }
    n0 += __shfl_xor_sync(0xffffffffu, n0, 1); n0 += __shfl_xor_sync(0xffffffffu, n0, 2);
    n1 += __shfl_xor_sync(0xffffffffu, n1, 1); n1 += __shfl_xor_sync(0xffffffffu, n1, 2);
    const float i0 = rsqrtf(fmaxf(n0, 1e-30f)), i1 = rsqrtf(fmaxf(n1, 1e-30f));
#pragma unroll
    for (int n = 0; n < NT; ++n) {
      const int q = 8 * n + 2 * t;
      const float s0 = s_inv[q], s1 = s_inv[q + 1];
      if (r0 < P) {
        if (q < Q) rel[r0 * Q + q] = c[n][0] * i0 * s0;
        if (q + 1 < Q) rel[r0 * Q + q + 1] = c[n][1] * i0 * s1;
      }
      if (r1 < P) {
        if (q < Q) rel[r1 * Q + q] = c[n][2] * i1 * s0;
        if (q + 1 < Q) rel[r1 * Q + q + 1] = c[n][3] * i1 * s1;
      }
    }
  }
}

}  // namespace

extern "C" int legs_relevancy_decoded(legs_ctx* ctx, const uint16_t* decoded, int64_t P, int32_t d, int32_t d_clip,
                                      const uint16_t* queries, int32_t Q, float* rel, void* stream) {
  if (!ctx) return LEGS_ERR_NULL;
  if (P < 0 || Q < 1 || Q > kMapQPad || d < 8 || (d & 7) || d_clip < 8 || (d_clip & 7) || d_clip > d || d_clip > 1024) return LEGS_ERR_DIM;
  if (!queries) return LEGS_ERR_NULL;
  if (P == 0) return LEGS_OK;
  if (!decoded || !rel) return LEGS_ERR_NULL;
  if (!legs_aligned16(decoded) || !legs_aligned16(queries) || !legs_aligned16(rel)) return LEGS_ERR_ALIGN;
  const int kblocks = (d_clip + 31) / 32;
  const int smem_bytes = kMapQPad * (kblocks * 64 + kMapRowPad) + kMapQPad * 4;   // <= 34 KB
  const long long tiles = (P + 15) / 16;
  const long long want = (tiles + kMapThreads / 32 - 1) / (kMapThreads / 32);
  const long long cap = (long long)ctx->num_sms * 8;
  const unsigned grid = (unsigned)(want < cap ? want : cap);
  cudaStream_t st = (cudaStream_t)stream;
  if (Q <= 8) relevancy_map_kernel<1><<<grid, kMapThreads, smem_bytes, st>>>(decoded, P, d, d_clip, queries, Q, rel);
  else relevancy_map_kernel<2><<<grid, kMapThreads, smem_bytes, st>>>(decoded, P, d, d_clip, queries, Q, rel);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

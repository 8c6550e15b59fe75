// forward.cu — S5: per-tile forward compositor (s_G is rendered "with rasterization and alpha
// blending" like colour, Eq. 8; :138: R_u likewise). Constants per BASELINE.json north_star (3) and readings C-9, C-10,
// C-13: alpha = min(0.99, o exp(power)), skip alpha < 1/255, stop before the Gaussian that would make T < 1e-4.
//
// One CTA per 16x16 tile, one thread per pixel; the tile's depth-ordered list is staged through shared memory in
// batches of 256 packed records (gathered by index). The exponent is evaluated through the scaled Cholesky factor of
// the conic kept in the record (common.cuh legs_pair_raw). FP32-ALU/MUFU bound.
#include "common.cuh"

namespace {

constexpr int kTileThreads = LEGS_TILE * LEGS_TILE;  // 256
constexpr float kAlphaMin = 1.0f / 255.0f;
constexpr float kAlphaMax = 0.99f;
constexpr float kTMin = 1e-4f;

// COUNT = true is the measurement variant (legs_render_forward_stats): same loop and same culling, plus work counters
// (pairs this kernel examines after block culling, blended pairs, staged list entries, and the pairs a plain
// per-tile walk without block culling would examine: every list entry up to the pixel's termination point).
// CTAs per SM: 4 at F <= 8 (64 registers), 3 at F <= 16 (80 registers), 2 beyond (128). Round 2 compiled every F > 8 for ONE
// CTA per SM (152 registers at F = 16: eight warps per SM); measured on configs[4] (F = 16, 3 M Gaussians, 1920x1080) the
// forward pass went 1.55 -> 0.98 ms with three. Four (64 registers, 48 bytes of spills) is slower again: 1.34 ms.
template <int F, bool COUNT>
__global__ void __launch_bounds__(kTileThreads, COUNT ? 1 : (F <= 8 ? 4 : F <= 16 ? 3 : 2)) forward_kernel(const uint32_t* __restrict__ vals,
                                                               const uint2* __restrict__ ranges,
                                                               const float* __restrict__ record, DevCamera cam,
                                                               float* __restrict__ out, uint32_t* __restrict__ n_contrib,
                                                               uint16_t* __restrict__ sem_bf16,
                                                               uint8_t* __restrict__ block_masks,
                                                               unsigned long long* __restrict__ counters) {
  constexpr int RS = (11 + F + 3) / 4 * 4;
  constexpr int CH = (6 + F + 3) / 4 * 4;
  constexpr int NV = F + 1;  // sem + unc
  // staged records + the head (32 bytes: all that is read before the alpha test) of a null record with opacity 0, the
  // padding entry of the candidate lists. Dynamic: 45 KB at F = 32.
  extern __shared__ __align__(16) float s_rec[];
  __shared__ uint32_t s_mask[kTileThreads];  // bit w: some pixel of warp w's 8x4 block can pass the alpha test
  __shared__ __align__(8) uint16_t s_cl[kTileThreads / 32][kTileThreads + 4];   // per warp: byte offsets of its candidates' records

  const int tile = cam.tile_order ? (int)cam.tile_order[blockIdx.x] : (int)blockIdx.x;   // heavy tiles first (legs_tile_order)
  const int tx = tile % cam.grid_x, ty = tile / cam.grid_x;
  int lx, ly;
  legs_tile_pixel(threadIdx.x, lx, ly);
  const int px = tx * LEGS_TILE + lx, py = ty * LEGS_TILE + ly;
  const bool inside = px < cam.width && py < cam.height;
  const uint2 rg = ranges[tile];
  const int count = (int)(rg.y - rg.x);
  // A pixel that has terminated (or lies outside the image) moves infinitely far away: every later pair evaluates to
  // alpha = 0 and is skipped by the alpha test, so the candidate loop needs no per-pixel "done" test and stays warp-uniform.
  constexpr float kFar = 3.0e18f;
  float fx = inside ? (float)px : kFar;
  const float fy = (float)py;

  float T = 1.0f;
  // accumulators in pairs (red, green), (blue, depth), (sem0, sem1), ..., (sem[F-2], sem[F-1]), (unc, -): the record keeps
  // the blended values in the same order, so every pair is one half of a 16-byte shared-memory load and one packed
  // fma.rn.f32x2 (two FP32 FMAs in one issue slot) updates it
  constexpr int NP = (4 + F + 2) / 2;   // (rgb, depth) 2 pairs + F/2 + (unc, pad)
  unsigned long long acc[NP];
#pragma unroll
  for (int k = 0; k < NP; ++k) acc[k] = 0ull;
  uint32_t last_off = 0;   // byte offset of the last blended record in its batch, and that batch's list base + 1
  int last_base = 0;       // (0: nothing blended)
  int done = inside ? 0 : 1;   // (an int: a bool gets byte-packed with other flags and costs PRMTs in the loop)
  uint32_t n_examined = 0, n_blended = 0, n_fetched = 0, n_plain = inside ? (uint32_t)count : 0u;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rec_base = legs_smem_addr(s_rec), cl_base = legs_smem_addr(&s_cl[warp][0]);
  if (threadIdx.x < 8) s_rec[kTileThreads * RS + threadIdx.x] = 0.f;
  for (int base = 0; base < count; base += kTileThreads) {
    if (__syncthreads_count(done) == kTileThreads) break;
    const int nb = min(kTileThreads, count - base);
    if (COUNT) n_fetched += nb;
    if ((int)threadIdx.x < nb) {
      const uint32_t g = vals[rg.x + base + threadIdx.x];
      const float4* src = reinterpret_cast<const float4*>(record + (size_t)g * RS);
      float4* dst = reinterpret_cast<float4*>(s_rec + threadIdx.x * RS);
      float4 q[RS / 4];
#pragma unroll
      for (int k = 0; k < RS / 4; ++k) { q[k] = src[k]; dst[k] = q[k]; }
      const uint32_t m = legs_block_mask(q[0].x, q[0].y, q[0].z, q[0].w, q[1].x, q[RS / 4 - 1].w, tx * LEGS_TILE,
                                         ty * LEGS_TILE);
      s_mask[threadIdx.x] = m;
      if (block_masks) block_masks[rg.x + base + threadIdx.x] = (uint8_t)m;   // kept for legs_render_backward
    }
    __syncthreads();
    if (__all_sync(0xffffffffu, done)) continue;
    // candidates of this warp's 8x4 block, front to back: compacted (one ballot per 32 list entries) into a list of record
    // offsets, padded to a multiple of four with the null record
    int ncand = 0;
    for (int c = 0; c * 32 < nb; ++c) {
      const int jl = c * 32 + lane;
      const bool is = jl < nb && ((s_mask[jl] >> warp) & 1u);
      const uint32_t m = __ballot_sync(0xffffffffu, is);
      if (is) s_cl[warp][ncand + __popc(m & ((1u << lane) - 1u))] = (uint16_t)(jl * (RS * 4));
      ncand += __popc(m);
    }
    if (lane < 4) s_cl[warp][ncand + lane] = (uint16_t)(kTileThreads * RS * 4);
    __syncwarp();
    for (int i0 = 0; i0 < ncand; i0 += 4) {
      const unsigned long long offs = legs_lds64_u64(cl_base + 2 * i0);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t off = (uint32_t)(offs >> (16 * k)) & 0xffffu;
        const uint32_t ra = rec_base + off;
        const float4 r0 = legs_lds128(ra);           // mu_x, mu_y, r11, r12
        const float2 r1lo = legs_lds64(ra + 16);     // r22, opacity
        float u, v;
        const float alpha = fminf(kAlphaMax, legs_pair_raw(fx, fy, r0, make_float4(r1lo.x, r1lo.y, 0.f, 0.f), u, v));
        if (COUNT && !done && off != (uint32_t)(kTileThreads * RS * 4)) ++n_examined;
        if (!(alpha < kAlphaMin)) {
          const float Tn = T * (1.0f - alpha);
          if (Tn < kTMin) {
            done = 1;
            fx = kFar;
            if (COUNT) n_plain = (uint32_t)base + off / (RS * 4) + 1u;
          } else {
            if (COUNT) ++n_blended;
            const float w = alpha * T;
            unsigned long long ww;
            asm("mov.b64 %0, {%1, %1};" : "=l"(ww) : "f"(w));
            // record floats 6.. : red, green | blue, depth | sem0, sem1 | ... | sem[F-2], sem[F-1] | unc, thr
            const unsigned long long q0 = legs_lds64_u64(ra + 24);   // (red, green)
            asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc[0]) : "l"(q0), "l"(ww));
#pragma unroll
            for (int kk = 0; kk < (F + 4) / 4; ++kk) {
              const ulonglong2 q = legs_lds128_u64(ra + 32 + 16 * kk);
              asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc[1 + 2 * kk]) : "l"(q.x), "l"(ww));
              asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc[2 + 2 * kk]) : "l"(q.y), "l"(ww));
            }
            T = Tn;
            last_off = off;
            last_base = base + 1;
          }
        }
      }
      if (__all_sync(0xffffffffu, done)) break;
    }
  }
  const uint32_t last = last_base ? (uint32_t)last_base + last_off / (RS * 4) : 0u;
  if (COUNT) {
    atomicAdd(&counters[0], (unsigned long long)n_examined);
    atomicAdd(&counters[1], (unsigned long long)n_blended);
    if (threadIdx.x == 0) atomicAdd(&counters[2], (unsigned long long)n_fetched);
    atomicAdd(&counters[3], (unsigned long long)n_plain);
  }
  if (inside) {
    const size_t p = (size_t)py * cam.width + px;
    float o[CH];
    float a[2 * NP];
#pragma unroll
    for (int k = 0; k < NP; ++k) asm("mov.b64 {%0, %1}, %2;" : "=f"(a[2 * k]), "=f"(a[2 * k + 1]) : "l"(acc[k]));
    // a: red, green, blue, depth, sem[F], unc, (thr-weighted pad: unused)
    o[0] = fmaf(T, cam.bg[0], a[0]); o[1] = fmaf(T, cam.bg[1], a[1]); o[2] = fmaf(T, cam.bg[2], a[2]);
    o[3] = a[3];
    float sv[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) { sv[k] = a[4 + k]; o[4 + k] = sv[k]; }
    o[5 + F] = 1.0f - T;
    o[6 + F] = T;  // final transmittance (kept for the backward pass: 1 - alpha loses it when T is small)
    o[7 + F] = 0.f;
    float4* dst = reinterpret_cast<float4*>(out + p * CH);
#pragma unroll
    for (int k = 0; k < CH / 4; ++k) dst[k] = make_float4(o[4 * k], o[4 * k + 1], o[4 * k + 2], o[4 * k + 3]);
    n_contrib[p] = last;
    if (sem_bf16) {
      uint32_t packed[F / 2];
#pragma unroll
      for (int k = 0; k < F / 2; ++k) {
        uint32_t u;
        asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(u) : "f"(sv[2 * k + 1]), "f"(sv[2 * k]));
        packed[k] = u;
      }
      uint4* d16 = reinterpret_cast<uint4*>(sem_bf16 + p * F);
#pragma unroll
      for (int k = 0; k < F / 8; ++k) d16[k] = make_uint4(packed[4 * k], packed[4 * k + 1], packed[4 * k + 2], packed[4 * k + 3]);
      if (F % 8) {
        uint2* d8 = reinterpret_cast<uint2*>(sem_bf16 + p * F + (F / 8) * 8);
        *d8 = make_uint2(packed[(F / 8) * 4], packed[(F / 8) * 4 + 1]);
      }
    }
  }
}

template <int F>
int launch_forward(legs_ctx* ctx, const DevCamera& dc, const legs_frame* frame, const uint32_t* vals,
                   const uint32_t* ranges, float* out, uint32_t* n_contrib, uint16_t* sem_bf16, uint8_t* block_masks,
                   unsigned long long* counters, cudaStream_t st) {
  const int ntiles = dc.grid_x * dc.grid_y;
  constexpr int RS = (11 + F + 3) / 4 * 4;
  constexpr size_t smem = (size_t)(kTileThreads * RS + 8) * sizeof(float);
  if (smem > 40 * 1024) {   // with the static arrays beyond the 48 KB a kernel gets without asking
    LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(forward_kernel<F, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(forward_kernel<F, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  }
  if (counters)
    forward_kernel<F, true><<<ntiles, kTileThreads, smem, st>>>(vals, (const uint2*)ranges, frame->record, dc, out, n_contrib,
                                                                sem_bf16, block_masks, counters);
  else
    forward_kernel<F, false><<<ntiles, kTileThreads, smem, st>>>(vals, (const uint2*)ranges, frame->record, dc, out,
                                                                 n_contrib, sem_bf16, block_masks, nullptr);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

}  // namespace

static int render_forward_impl(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam, const legs_frame* frame,
                               const uint32_t* vals_sorted, const uint32_t* ranges, float* out_pixels,
                               uint32_t* n_contrib, uint16_t* sem_bf16, uint8_t* block_masks,
                               unsigned long long* counters, void* stream, const uint32_t* tile_order = nullptr) {
  if (!ctx) return LEGS_ERR_NULL;
  if (tile_order && !legs_aligned16(tile_order)) return LEGS_ERR_ALIGN;
  int rc;
  if ((rc = legs_check_gaussians(g)) != LEGS_OK) return rc;
  if ((rc = legs_check_camera(cam)) != LEGS_OK) return rc;
  if ((rc = legs_check_frame(frame)) != LEGS_OK) return rc;
  if (!vals_sorted || !ranges || !out_pixels || !n_contrib) return LEGS_ERR_NULL;
  if (!legs_aligned16(vals_sorted) || !legs_aligned16(ranges) || !legs_aligned16(out_pixels) ||
      !legs_aligned16(n_contrib) || (sem_bf16 && !legs_aligned16(sem_bf16)))
    return LEGS_ERR_ALIGN;
  DevCamera dc = make_dev_camera(cam);
  dc.tile_order = tile_order;
  cudaStream_t st = (cudaStream_t)stream;
#define LEGS_FWD_CASE(FF) \
  case FF: return launch_forward<FF>(ctx, dc, frame, vals_sorted, ranges, out_pixels, n_contrib, sem_bf16, block_masks, counters, st);
  switch (g->sem_dim) {
    LEGS_FWD_CASE(4) LEGS_FWD_CASE(8) LEGS_FWD_CASE(12) LEGS_FWD_CASE(16) LEGS_FWD_CASE(20) LEGS_FWD_CASE(24)
    LEGS_FWD_CASE(28) LEGS_FWD_CASE(32)
    default: return LEGS_ERR_DIM;
  }
#undef LEGS_FWD_CASE
}

extern "C" int legs_render_forward(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam,
                                   const legs_frame* frame, const uint32_t* vals_sorted, const uint32_t* ranges,
                                   float* out_pixels, uint32_t* n_contrib, uint16_t* sem_bf16, uint8_t* block_masks,
                                   void* stream) {
  return render_forward_impl(ctx, g, cam, frame, vals_sorted, ranges, out_pixels, n_contrib, sem_bf16, block_masks, nullptr,
                             stream);
}

extern "C" int legs_render_forward_ordered(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam,
                                           const legs_frame* frame, const uint32_t* vals_sorted, const uint32_t* ranges,
                                           float* out_pixels, uint32_t* n_contrib, uint16_t* sem_bf16, uint8_t* block_masks,
                                           const uint32_t* tile_order, void* stream) {
  return render_forward_impl(ctx, g, cam, frame, vals_sorted, ranges, out_pixels, n_contrib, sem_bf16, block_masks, nullptr,
                             stream, tile_order);
}

extern "C" int legs_render_forward_stats(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam,
                                         const legs_frame* frame, const uint32_t* vals_sorted, const uint32_t* ranges,
                                         float* out_pixels, uint32_t* n_contrib, uint64_t* counters, void* stream) {
  if (!counters) return LEGS_ERR_NULL;
  if (!legs_aligned16(counters)) return LEGS_ERR_ALIGN;
  return render_forward_impl(ctx, g, cam, frame, vals_sorted, ranges, out_pixels, n_contrib, nullptr, nullptr,
                             (unsigned long long*)counters, stream);
}

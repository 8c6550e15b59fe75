// backward.cu — S6: back-to-front backward compositor (BASELINE.json north_star (4); "differentiable
// rendering", :182). Per pixel, contributors k = last..first:
//   dL/dv_k,ch += w_k G_ch;   dL/dalpha_k = sum_ch G_ch (T_k v_k,ch - S_ch/(1-alpha_k)),
// the channel sum over rgb only unless LEGS_BWD_COUPLE_SEM (reading C-14); zero through the 0.99 clamp (C-15).
// The suffix S_ch is carried in the normalised form A_ch = (sum_{j>k} w_j v_j,ch) / T_{k+1}, A <- alpha v + (1-alpha) A.
//
// Geometry sums are taken in the whitened coordinates (u, v) = R' (pixel - mean) of the record (R' = scaled Cholesky
// factor of the conic, preprocess.cu): with dpow = dL/dpower the kernel accumulates per Gaussian
//   S0 = sum dpow,  (Su, Sv) = sum dpow (u, v),  (Huu, Huv, Hvv) = sum dpow (u^2, u v, v^2)
// from which project_backward.cu forms dL/dopacity = S0 / o, dL/dmu = R^T (Su, Sv) and dL/dSigma' = 1/2 R^T H R.
// That is the same gradient as the (A, B, C) form of DESIGN.md section 2 (H = R G_d R^T with G_d = sum dpow d d^T, and
// -Q dQ Q = 1/2 Q G_d Q = 1/2 R^T H R), with bounded factors (u^2 + v^2 <= log2(255 o)) in place of dx^2 ~ 1e4 and no
// ill-conditioned Q dQ Q product afterwards, so fp32 atomics suffice.
//
// Reduction: the 10+F per-Gaussian partial sums of a warp's 32 pixels (an 8x4 block) are reduced with a compact
// butterfly transpose (20 shuffles for 18 values instead of 5 per value), after which each lane owns one value and
// issues one red.global.add for it into the Gaussian's row of the scratch array. The first two rounds of the channel
// values need no selects: every lane keeps its upstream gradients G in the register order its own path through the
// butterfly wants (a per-lane permutation fixed by lane bits 4 and 3, applied once per tile when G is loaded).
#include "common.cuh"

namespace {

constexpr int kTileThreads = LEGS_TILE * LEGS_TILE;
constexpr float kAlphaMin = 1.0f / 255.0f;
constexpr float kAlphaMax = 0.99f;

// One butterfly round over the first N entries of v (xor offset OFF): N -> ceil(N/2) live values; lanes with the
// offset bit set keep the upper half. Lanes whose path runs through padding hold exact zeros.
template <int N, int OFF, int NVMAX>
__device__ __forceinline__ void bfly_round(float (&v)[NVMAX], int lane) {
  constexpr int H = (N + 1) / 2;
  const bool upper = (lane & OFF) != 0;
#pragma unroll
  for (int i = 0; i < H; ++i) {
    const float hi = (i + H < N) ? v[i + H] : 0.f;
    const float send = upper ? v[i] : hi;
    const float keep = upper ? hi : v[i];
    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, OFF);
  }
}
// Select-free round for values whose register order was permuted per lane beforehand: everybody keeps [0, N/2) and
// sends [N/2, N).
template <int N, int OFF, int NVMAX>
__device__ __forceinline__ void bfly_round_baked(float (&v)[NVMAX]) {
  static_assert(N % 2 == 0, "baked rounds need an even count");
#pragma unroll
  for (int i = 0; i < N / 2; ++i) v[i] += __shfl_xor_sync(0xffffffffu, v[i + N / 2], OFF);
}

// Index bookkeeping of the reduction (all compile-time in F, run-time in the lane id).
// GEO (LEGS_BWD_DEPTH_ALPHA, reading C-17b): the depth image has an upstream gradient too, so depth is one more blended
// channel: the channel list becomes rgb[3], depth, sem[F], unc (= the order of the pixel record and of the Gaussian
// record), padded with zero channels to a multiple of 4.
template <int F, bool GEO>
struct Red {
  static constexpr int NCR = GEO ? 3 + 1 + F + 1 : 3 + F + 1;   // real channels
  static constexpr int NC = (NCR + 3) / 4 * 4;                  // channel values: drgb[3], (ddepth,) dsem[F], dunc (, padding)
  // slot of channel c in the pixel record (and, + 6, in the Gaussian record)
  __device__ static __forceinline__ constexpr int pix_slot(int c) { return GEO ? c : (c < 3 ? c : c + 1); }
  static constexpr int Q = NC / 4;          // channel values left per lane after the two baked rounds
  static constexpr int M = 2 + Q;           // merged list for the rounds with offsets 4, 2, 1: 2 geometry + Q channel
  static constexpr int m1 = (M + 1) / 2, m2 = (m1 + 1) / 2, m3 = (m2 + 1) / 2;
  static constexpr int NOUT = m3;           // values a lane owns at the end
  static_assert(NC % 4 == 0 && NOUT <= 2, "F is a multiple of 4, at most 32");
  static constexpr int RG = (6 + NC + 3) / 4 * 4;   // floats per Gaussian row of the scratch array
  // channel held in register i of the permuted array by this lane
  __device__ static __forceinline__ int channel_of(int i, int lane) {
    const int b = i / (NC / 2), within = i % (NC / 2), hb = within / Q, j = within % Q;
    return (NC / 2) * (((lane >> 4) & 1) ^ b) + Q * (((lane >> 3) & 1) ^ hb) + j;
  }
  // output slot (0 S0, 1 Su, 2 Sv, 3 Huu, 4 Huv, 5 Hvv, 6.. channels) of merged-list entry t for this lane; -1 = padding
  __device__ static __forceinline__ int slot_of_merged(int t, int lane) {
    if (t >= M) return -1;
    const int b4 = (lane >> 4) & 1, b3 = (lane >> 3) & 1;
    if (t == 0) return 3 * b4 + 2 * b3;
    if (t == 1) return b3 ? -1 : 3 * b4 + 1;
    return 6 + (NC / 2) * b4 + Q * b3 + (t - 2);
  }
  // first merged-list index this lane owns after the rounds with offsets 4, 2, 1
  __device__ static __forceinline__ int merged_index(int lane) {
    return ((lane >> 2) & 1) * m1 + ((lane >> 1) & 1) * m2 + (lane & 1) * m3;
  }
};

// MASKS: the per-entry warp-block masks come from the forward pass (block_masks); otherwise they are recomputed here
// (a separate instantiation: the recomputation costs registers the hot loop should not pay for).
template <int F, bool COUPLE, bool MASKS, bool GEO>
__global__ void __launch_bounds__(kTileThreads) backward_kernel(const uint32_t* __restrict__ vals,
                                                                const uint2* __restrict__ ranges,
                                                                const float* __restrict__ record, DevCamera cam,
                                                                const float* __restrict__ out_pixels,
                                                                const uint32_t* __restrict__ n_contrib,
                                                                const float* __restrict__ dL_dpix,
                                                                const uint8_t* __restrict__ block_masks,
                                                                float* __restrict__ gscr) {
  constexpr int RS = (11 + F + 3) / 4 * 4;
  constexpr int CH = (6 + F + 3) / 4 * 4;
  using R = Red<F, GEO>;
  constexpr int RG = R::RG;
  constexpr int NC = R::NC;
  constexpr int NA = COUPLE ? R::NCR : (GEO ? 4 : 3);  // channels whose suffix sums feed dL/dalpha
  __shared__ __align__(16) float s_rec[kTileThreads * RS];
  __shared__ uint32_t s_idx[kTileThreads];
  __shared__ uint8_t s_mask[kTileThreads];   // bit w: some pixel of warp w's 8x4 block can pass the alpha test
  __shared__ uint8_t s_cl[kTileThreads / 32][kTileThreads];   // per warp: its candidates of the batch (list positions)
  __shared__ int s_max;

  const int tile = cam.tile_order ? (int)cam.tile_order[blockIdx.x] : (int)blockIdx.x;   // heavy tiles first (legs_tile_order)
  const int tx = tile % cam.grid_x, ty = tile / cam.grid_x;
  int lx, ly;
  legs_tile_pixel(threadIdx.x, lx, ly);
  const int px = tx * LEGS_TILE + lx, py = ty * LEGS_TILE + ly;
  const bool inside = px < cam.width && py < cam.height;
  const int lane = threadIdx.x & 31;
  const uint2 rg = ranges[tile];
  const float fx = (float)px, fy = (float)py;

  float G[NA], A[NA];
  unsigned long long Gpp[NC / 2];   // upstream gradients in this lane's butterfly order, as packed pairs
  float T = 1.f;
  int ncon = 0;
  if (inside) {
    const size_t p = (size_t)py * cam.width + px;
    const float* grow = dL_dpix + p * CH;
#pragma unroll
    for (int k = 0; k < NA; ++k) G[k] = grow[R::pix_slot(k)];
#pragma unroll
    for (int i = 0; i < NC / 2; ++i) {   // the same gradients in this lane's butterfly order
      const int c0 = R::channel_of(2 * i, lane), c1 = R::channel_of(2 * i + 1, lane);
      const float g0 = c0 < R::NCR ? grow[R::pix_slot(c0)] : 0.f, g1 = c1 < R::NCR ? grow[R::pix_slot(c1)] : 0.f;
      asm("mov.b64 %0, {%1, %2};" : "=l"(Gpp[i]) : "f"(g0), "f"(g1));
    }
    T = out_pixels[p * CH + 6 + F];
    ncon = (int)n_contrib[p];
  } else {
#pragma unroll
    for (int k = 0; k < NA; ++k) G[k] = 0.f;
#pragma unroll
    for (int i = 0; i < NC / 2; ++i) Gpp[i] = 0ull;
  }
#pragma unroll
  for (int k = 0; k < NA; ++k) A[k] = 0.f;
  // background term: d(T_final * bg)/dalpha_k = -T_final bg / (1 - alpha_k); the alpha image 1 - T_final is the same form
  // with a "background" of -1 (GEO)
  float bgG = inside ? T * (cam.bg[0] * G[0] + cam.bg[1] * G[1] + cam.bg[2] * G[2]) : 0.f;
  if (GEO && inside) bgG = fmaf(-T, dL_dpix[((size_t)py * cam.width + px) * CH + 5 + F], bgG);

  if (threadIdx.x == 0) s_max = 0;
  __syncthreads();
  int wmax = ncon;  // last list position any pixel of this warp blended
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, off));
  if (lane == 0) atomicMax(&s_max, wmax);
  __syncthreads();
  const int maxc = s_max;
  const int warp = threadIdx.x >> 5;

  // scratch slot(s) this lane owns after the butterfly (-1: none)
  int my_slot[R::NOUT];
#pragma unroll
  for (int j = 0; j < R::NOUT; ++j) my_slot[j] = R::slot_of_merged(R::merged_index(lane) + j, lane);

  const uint32_t rec_base = legs_smem_addr(s_rec), idx_base = legs_smem_addr(s_idx);
  const int nbatches = (maxc + kTileThreads - 1) / kTileThreads;
  for (int b = nbatches - 1; b >= 0; --b) {
    const int base = b * kTileThreads;
    const int nb = min(kTileThreads, maxc - base);
    __syncthreads();
    if ((int)threadIdx.x < nb) {
      const uint32_t g = vals[rg.x + base + threadIdx.x];
      s_idx[threadIdx.x] = g;
      const float4* src = reinterpret_cast<const float4*>(record + (size_t)g * RS);
      float4* dst = reinterpret_cast<float4*>(s_rec + threadIdx.x * RS);
      float4 q[RS / 4];
#pragma unroll
      for (int k = 0; k < RS / 4; ++k) { q[k] = src[k]; dst[k] = q[k]; }
      // the forward pass computed the same mask for this list entry; reuse it when the caller kept it
      s_mask[threadIdx.x] = MASKS ? block_masks[rg.x + base + threadIdx.x]
                                  : (uint8_t)legs_block_mask(q[0].x, q[0].y, q[0].z, q[0].w, q[1].x, q[RS / 4 - 1].w, tx * LEGS_TILE,
                                                    ty * LEGS_TILE);
    }
    __syncthreads();
    // candidates of this warp: compacted, one ballot per 32 list entries, into a list that is then walked back to front
    // (warp-uniform: no per-lane candidate masks)
    const int lim = min(nb, wmax - base);
    int ncand = 0;
    for (int c = 0; c * 32 < lim; ++c) {
      const int jl = c * 32 + lane;
      const bool is = jl < lim && ((s_mask[jl] >> warp) & 1u);
      const uint32_t mm = __ballot_sync(0xffffffffu, is);
      if (is) s_cl[warp][ncand + __popc(mm & ((1u << lane) - 1u))] = (uint8_t)jl;
      ncand += __popc(mm);
    }
    __syncwarp();
    const int nrel = ncon - base;   // list positions below this (relative to the batch) were blended by this pixel
    {
      for (int i = ncand - 1; i >= 0; --i) {
        const int j = (int)s_cl[warp][i];
        const uint32_t ra = rec_base + (uint32_t)j * (RS * 4);
        const float4 r0 = legs_lds128(ra);        // mu_x, mu_y, r11, r12
        const float4 r1 = legs_lds128(ra + 16);   // r22, opacity, red, green
        float u, v;
        const float raw = legs_pair_raw(fx, fy, r0, r1, u, v);
        const float alpha = fminf(kAlphaMax, raw);
        const bool contrib = (j < nrel) && !(alpha < kAlphaMin);
        if (!__any_sync(0xffffffffu, contrib)) continue;
        // branch-free from here on: lanes that do not contribute carry alpha = 0 (w = 0, A and T unchanged)
        const float al = contrib ? alpha : 0.f;
        const float om = 1.0f - al;
        // 1 / om for om in [0.01, 1]: MUFU.RCP + one Newton step (branch-free)
        float rcp;
        asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rcp) : "f"(om));
        rcp = fmaf(rcp, fmaf(-om, rcp, 1.0f), rcp);
        T *= rcp;  // transmittance in front of this Gaussian
        const float w = al * T;
        // blended values of the channels in the dL/dalpha sum: record floats 6.. = red, green, blue, depth, sem[F], u
        constexpr int NV = R::pix_slot(NA - 1) + 1;
        float rv[(NV + 1) / 4 * 4 + 2];
        rv[0] = r1.z; rv[1] = r1.w;
#pragma unroll
        for (int k = 2; k < NV; k += 4) {
          const float4 q = legs_lds128(ra + (6 + k) * 4);
          rv[k] = q.x; rv[k + 1] = q.y; rv[k + 2] = q.z; rv[k + 3] = q.w;
        }
        float val[NA];
#pragma unroll
        for (int k = 0; k < NA; ++k) val[k] = rv[R::pix_slot(k)];
        float dLda = 0.f;
#pragma unroll
        for (int k = 0; k < NA; ++k) {
          const float d = val[k] - A[k];
          dLda = fmaf(G[k], d, dLda);
          A[k] = fmaf(al, d, A[k]);  // alpha*v + (1-alpha)*A
        }
        dLda = fmaf(dLda, T, -bgG * rcp);
        // zero through the 0.99 clamp (C-15) and for lanes that do not contribute
        const float dLdg = (contrib && !(raw > kAlphaMax)) ? dLda : 0.f;
        const float dpow = raw * dLdg;
        float geo[6];
        geo[0] = dpow;
        geo[1] = dpow * u;
        geo[2] = dpow * v;
        geo[3] = geo[1] * u;
        geo[4] = geo[1] * v;
        geo[5] = geo[2] * v;
        // channel values w * G in pairs: one packed multiply (mul.rn.f32x2: two FP32 products in one issue slot) per
        // pair, and the first select-free round adds pairs too
        float ch[NC / 2];
        {
          unsigned long long ww, hi[NC / 4], lo[NC / 4];
          asm("mov.b64 %0, {%1, %1};" : "=l"(ww) : "f"(w));
#pragma unroll
          for (int i = 0; i < NC / 4; ++i) {
            asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(lo[i]) : "l"(Gpp[i]), "l"(ww));
            asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(hi[i]) : "l"(Gpp[i + NC / 4]), "l"(ww));
          }
#pragma unroll
          for (int i = 0; i < NC / 4; ++i) {
            float h0, h1;
            asm("mov.b64 {%0, %1}, %2;" : "=f"(h0), "=f"(h1) : "l"(hi[i]));
            h0 = __shfl_xor_sync(0xffffffffu, h0, 16);
            h1 = __shfl_xor_sync(0xffffffffu, h1, 16);
            unsigned long long rcv;
            asm("mov.b64 %0, {%1, %2};" : "=l"(rcv) : "f"(h0), "f"(h1));
            asm("add.rn.f32x2 %0, %0, %1;" : "+l"(lo[i]) : "l"(rcv));
            asm("mov.b64 {%0, %1}, %2;" : "=f"(ch[2 * i]), "=f"(ch[2 * i + 1]) : "l"(lo[i]));
          }
        }
        // rounds with offsets 16 and 8: geometry with selects (6 -> 3 -> 2), channels without (NC -> NC/2 -> NC/4)
        bfly_round<6, 16, 6>(geo, lane);
        bfly_round<3, 8, 6>(geo, lane);
        bfly_round_baked<NC / 2, 8, NC / 2>(ch);
        float m[R::M];
        m[0] = geo[0]; m[1] = geo[1];
#pragma unroll
        for (int i = 0; i < R::Q; ++i) m[2 + i] = ch[i];
        bfly_round<R::M, 4, R::M>(m, lane);
        bfly_round<R::m1, 2, R::M>(m, lane);
        bfly_round<R::m2, 1, R::M>(m, lane);
        float* row = gscr + (size_t)legs_lds32(idx_base + 4 * j) * RG;
#pragma unroll
        for (int q = 0; q < R::NOUT; ++q)
          if (my_slot[q] >= 0 && m[q] != 0.f) atomicAdd(row + my_slot[q], m[q]);
      }
    }
  }
}

template <int F, bool GEO>
int launch_backward(legs_ctx* ctx, const DevCamera& dc, const legs_frame* frame, const uint32_t* vals,
                    const uint32_t* ranges, const float* out_pixels, const uint32_t* n_contrib, const float* dL,
                    const uint8_t* block_masks, int couple, float* o, cudaStream_t st) {
  const int ntiles = dc.grid_x * dc.grid_y;
#define LEGS_BWD_LAUNCH(C, M)                                                                                          \
  backward_kernel<F, C, M, GEO><<<ntiles, kTileThreads, 0, st>>>(vals, (const uint2*)ranges, frame->record, dc,       \
                                                                out_pixels, n_contrib, dL, block_masks, o)
  if (couple) { if (block_masks) LEGS_BWD_LAUNCH(true, true); else LEGS_BWD_LAUNCH(true, false); }
  else        { if (block_masks) LEGS_BWD_LAUNCH(false, true); else LEGS_BWD_LAUNCH(false, false); }
#undef LEGS_BWD_LAUNCH
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

}  // namespace

// defined in project_backward.cu
int legs_project_backward_launch(legs_ctx* ctx, const legs_gaussians* g, const DevCamera& dc, const legs_frame* frame,
                                 const float* gscr, legs_grads* grads, int accumulate, int geo, cudaStream_t st);

// floats per Gaussian row of the scratch array: S0, Su, Sv, Huu, Huv, Hvv, then the channel sums (see Red)
static size_t scratch_row_floats(int sem_dim, bool geo) {
  const int ncr = geo ? sem_dim + 5 : sem_dim + 4;
  return (size_t)((6 + (ncr + 3) / 4 * 4 + 3) / 4 * 4);
}

extern "C" {

size_t legs_backward_workspace_bytes(int64_t n, int32_t sem_dim) {
  // one row per Gaussian: the sums the compositor reduces (see the head of this file); sized for the wider row of
  // LEGS_BWD_DEPTH_ALPHA
  const size_t nn = (size_t)(n > 0 ? n : 1);
  return legs_align_up(nn * scratch_row_floats(sem_dim > 0 ? sem_dim : 0, true) * 4, 256);
}

int legs_render_backward(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam, const legs_frame* frame,
                         const uint32_t* vals_sorted, const uint32_t* ranges, const float* out_pixels,
                         const uint32_t* n_contrib, const float* dL_dpixels, const uint8_t* block_masks, int32_t flags,
                         legs_grads* grads, void* workspace, size_t workspace_bytes, void* stream) {
  return legs_render_backward_ordered(ctx, g, cam, frame, vals_sorted, ranges, out_pixels, n_contrib, dL_dpixels, block_masks,
                                      flags, grads, workspace, workspace_bytes, nullptr, stream);
}

int legs_render_backward_ordered(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam, const legs_frame* frame,
                                 const uint32_t* vals_sorted, const uint32_t* ranges, const float* out_pixels,
                                 const uint32_t* n_contrib, const float* dL_dpixels, const uint8_t* block_masks,
                                 int32_t flags, legs_grads* grads, void* workspace, size_t workspace_bytes,
                                 const uint32_t* tile_order, void* stream) {
  if (!ctx) return LEGS_ERR_NULL;
  if (tile_order && !legs_aligned16(tile_order)) return LEGS_ERR_ALIGN;
  int rc;
  if ((rc = legs_check_gaussians(g)) != LEGS_OK) return rc;
  if ((rc = legs_check_camera(cam)) != LEGS_OK) return rc;
  if ((rc = legs_check_frame(frame)) != LEGS_OK) return rc;
  if (!vals_sorted || !ranges || !out_pixels || !n_contrib || !dL_dpixels || !grads || !workspace) return LEGS_ERR_NULL;
  if (!grads->dmeans || !grads->dscales || !grads->dquats || !grads->dopacities || !grads->dsh || !grads->dsem ||
      !grads->dunc || !grads->dmean2d)
    return LEGS_ERR_NULL;
  if (!legs_aligned16(vals_sorted) || !legs_aligned16(ranges) || !legs_aligned16(out_pixels) ||
      !legs_aligned16(n_contrib) || !legs_aligned16(dL_dpixels) || !legs_aligned16(workspace) ||
      !legs_aligned16(grads->dmeans) || !legs_aligned16(grads->dscales) || !legs_aligned16(grads->dquats) ||
      !legs_aligned16(grads->dopacities) || !legs_aligned16(grads->dsh) || !legs_aligned16(grads->dsem) ||
      !legs_aligned16(grads->dunc) || !legs_aligned16(grads->dmean2d))
    return LEGS_ERR_ALIGN;
  if (workspace_bytes < legs_backward_workspace_bytes(g->n, g->sem_dim)) return LEGS_ERR_WORKSPACE;
  if (g->n == 0) return LEGS_OK;
  cudaStream_t st = (cudaStream_t)stream;
  const int F = g->sem_dim;
  const bool acc = (flags & LEGS_BWD_ACCUMULATE) != 0;
  float* o = (float*)workspace;
  const bool geo = (flags & LEGS_BWD_DEPTH_ALPHA) != 0;
  LEGS_CUDA_CHECK(ctx, cudaMemsetAsync(o, 0, (size_t)g->n * scratch_row_floats(F, geo) * 4, st));
  DevCamera dc = make_dev_camera(cam);
  dc.tile_order = tile_order;
  const int couple = (flags & LEGS_BWD_COUPLE_SEM) ? 1 : 0;
#define LEGS_BWD_CASE(FF)                                                                                            \
  case FF:                                                                                                           \
    rc = geo ? launch_backward<FF, true>(ctx, dc, frame, vals_sorted, ranges, out_pixels, n_contrib, dL_dpixels,         \
                                         block_masks, couple, o, st)                                                    \
             : launch_backward<FF, false>(ctx, dc, frame, vals_sorted, ranges, out_pixels, n_contrib, dL_dpixels,        \
                                          block_masks, couple, o, st);                                                   \
    break;
  switch (F) {
    LEGS_BWD_CASE(4) LEGS_BWD_CASE(8) LEGS_BWD_CASE(12) LEGS_BWD_CASE(16) LEGS_BWD_CASE(20) LEGS_BWD_CASE(24)
    LEGS_BWD_CASE(28) LEGS_BWD_CASE(32)
    default: return LEGS_ERR_DIM;
  }
#undef LEGS_BWD_CASE
  if (rc != LEGS_OK) return rc;
  if (flags & LEGS_BWD_COMPOSITE_ONLY) return LEGS_OK;   // measurement: S6 alone (grads are not written)
  return legs_project_backward_launch(ctx, g, dc, frame, o, grads, acc ? 1 : 0, geo ? 1 : 0, st);
}

}  // extern "C"

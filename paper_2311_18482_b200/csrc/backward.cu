// backward.cu — S6: back-to-front backward compositor (BASELINE.json north_star (4); "differentiable
// rendering", :182). Per pixel, contributors k = last..first:
//   dL/dv_k,ch += w_k G_ch;   dL/dalpha_k = sum_ch G_ch (T_k v_k,ch - S_ch/(1-alpha_k)),
// the channel sum over rgb only unless LEGS_BWD_COUPLE_SEM (reading C-14); zero through the 0.99 clamp (C-15).
// The suffix S_ch is carried in the normalised form A_ch = (sum_{j>k} w_j v_j,ch) / T_{k+1}, A <- alpha v + (1-alpha) A.
//
// Reduction: the 10+F per-Gaussian partial sums of a warp's 32 pixels (an 8x4 block) are reduced with a compact
// butterfly transpose (20 shuffles for 18 values instead of 5 per value), after which each lane owns one value and
// issues one red.global.add for it.
#include "common.cuh"

namespace {

constexpr int kTileThreads = LEGS_TILE * LEGS_TILE;
constexpr float kAlphaMin = 1.0f / 255.0f;
constexpr float kAlphaMax = 0.99f;

// Compact butterfly transpose-reduction of NV per-lane values over the 32 lanes of a warp: round r (xor offset
// 16, 8, 4, 2, 1) halves the number of live values per lane (n -> ceil(n/2)); lanes with the offset bit set keep the
// upper half. sum_r ceil-halvings = 20 shuffles for NV = 18 instead of 5 per value. Afterwards lane l holds, in
// v[0..ceil(NV/32)-1], the warp totals of the values slot(l) + j with slot(l) = sum_r bit_r(l) * half_r; lanes whose
// path ran through padding hold exact zeros.
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

template <int NV>
struct Bfly {
  static constexpr int c1 = (NV + 1) / 2, c2 = (c1 + 1) / 2, c3 = (c2 + 1) / 2, c4 = (c3 + 1) / 2, c5 = (c4 + 1) / 2;
  static_assert(c5 <= 2, "at most 64 values");
  __device__ static __forceinline__ void reduce(float (&v)[NV], int lane) {
    bfly_round<NV, 16, NV>(v, lane);
    bfly_round<c1, 8, NV>(v, lane);
    bfly_round<c2, 4, NV>(v, lane);
    bfly_round<c3, 2, NV>(v, lane);
    bfly_round<c4, 1, NV>(v, lane);
  }
  __device__ static __forceinline__ int slot(int lane) {
    return ((lane >> 4) & 1) * c1 + ((lane >> 3) & 1) * c2 + ((lane >> 2) & 1) * c3 + ((lane >> 1) & 1) * c4 + (lane & 1) * c5;
  }
};

struct BwdOut {
  float* dopac;    // [n]
  float* dmean2d;  // [n,2]
  double* dconic;  // [n,3] scratch, fp64: thousands of near-cancelling per-warp partial sums meet here (G-4)
  float* drgb;     // [n,3] scratch
  float* dsem;     // [n,F]
  float* dunc;     // [n]
};

// value slots: 0 dopac, 1-2 dmean2d, 3-5 dconic, 6-8 drgb, 9..9+F-1 dsem, 9+F dunc
template <int F>
__device__ __forceinline__ void slot_address(const BwdOut& o, int slot, float*& base, int& stride) {
  base = nullptr; stride = 0;
  if (slot == 0) { base = o.dopac; stride = 1; }
  else if (slot < 3) { base = o.dmean2d + (slot - 1); stride = 2; }
  else if (slot < 6) { base = nullptr; stride = 3; }  // dconic: fp64 scratch, addressed separately
  else if (slot < 9) { base = o.drgb + (slot - 6); stride = 3; }
  else if (slot < 9 + F) { base = o.dsem + (slot - 9); stride = F; }
  else if (slot == 9 + F) { base = o.dunc; stride = 1; }
}

template <int F, bool COUPLE>
__global__ void __launch_bounds__(kTileThreads) backward_kernel(const uint32_t* __restrict__ vals,
                                                                const uint2* __restrict__ ranges,
                                                                const float* __restrict__ record, DevCamera cam,
                                                                const float* __restrict__ out_pixels,
                                                                const uint32_t* __restrict__ n_contrib,
                                                                const float* __restrict__ dL_dpix, BwdOut o) {
  constexpr int RS = (11 + F + 3) / 4 * 4;
  constexpr int CH = (6 + F + 3) / 4 * 4;
  constexpr int NC = 3 + F + 1;  // blended channels with an upstream gradient: rgb, sem, unc
  constexpr int NA = COUPLE ? NC : 3;  // channels whose suffix sums feed dL/dalpha
  constexpr int NV = 10 + F;
  constexpr int NOUT = (NV + 31) / 32;
  __shared__ __align__(16) float s_rec[kTileThreads * RS];
  __shared__ uint32_t s_idx[kTileThreads];
  __shared__ uint32_t s_mask[kTileThreads];  // bit w: some pixel of warp w's 8x4 block can pass the alpha test
  __shared__ int s_max;

  const int tile = blockIdx.x;
  const int tx = tile % cam.grid_x, ty = tile / cam.grid_x;
  int lx, ly;
  legs_tile_pixel(threadIdx.x, lx, ly);
  const int px = tx * LEGS_TILE + lx, py = ty * LEGS_TILE + ly;
  const bool inside = px < cam.width && py < cam.height;
  const int lane = threadIdx.x & 31;
  const uint2 rg = ranges[tile];
  const float fx = (float)px, fy = (float)py;

  float G[NC], A[NA];
  float T = 1.f;
  int ncon = 0;
  if (inside) {
    const size_t p = (size_t)py * cam.width + px;
    const float4* g4 = reinterpret_cast<const float4*>(dL_dpix + p * CH);
    float g[CH];
#pragma unroll
    for (int k = 0; k < CH / 4; ++k) {
      const float4 q = g4[k];
      g[4 * k] = q.x; g[4 * k + 1] = q.y; g[4 * k + 2] = q.z; g[4 * k + 3] = q.w;
    }
    G[0] = g[0]; G[1] = g[1]; G[2] = g[2];
#pragma unroll
    for (int k = 0; k < F + 1; ++k) G[3 + k] = g[4 + k];
    T = out_pixels[p * CH + 6 + F];
    ncon = (int)n_contrib[p];
  } else {
#pragma unroll
    for (int k = 0; k < NC; ++k) G[k] = 0.f;
  }
#pragma unroll
  for (int k = 0; k < NA; ++k) A[k] = 0.f;
  // background term: d(T_final * bg)/dalpha_k = -T_final bg / (1 - alpha_k)
  const float bgG = inside ? T * (cam.bg[0] * G[0] + cam.bg[1] * G[1] + cam.bg[2] * G[2]) : 0.f;

  if (threadIdx.x == 0) s_max = 0;
  __syncthreads();
  int wmax = ncon;  // last list position any pixel of this warp blended
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, off));
  if (lane == 0) atomicMax(&s_max, wmax);
  __syncthreads();
  const int maxc = s_max;
  const int warp = threadIdx.x >> 5;

  // output address of the value(s) this lane owns after the butterfly
  float* my_base[NOUT]; int my_stride[NOUT];
#pragma unroll
  for (int j = 0; j < NOUT; ++j) {
    const int sl = Bfly<NV>::slot(lane) + j;
    my_base[j] = nullptr; my_stride[j] = 0;
    if (sl < NV) slot_address<F>(o, sl, my_base[j], my_stride[j]);
  }
  const int sl0 = Bfly<NV>::slot(lane);   // slots 3..5 (dconic) always land in v[0]: NV >= 14 > 5 + 32 * 0
  double* my_conic = (sl0 >= 3 && sl0 < 6) ? o.dconic + (sl0 - 3) : nullptr;

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
      s_mask[threadIdx.x] = legs_block_mask(q[0].x, q[0].y, q[0].z, q[0].w, q[1].x, q[RS / 4 - 1].w, tx * LEGS_TILE, ty * LEGS_TILE);
    }
    __syncthreads();
    // candidates of this warp, back to front: 32 list entries at a time, one ballot each
    const int lim = min(nb, wmax - base);
    for (int c = (lim - 1) >> 5; c >= 0; --c) {
    const int jl = c * 32 + lane;
    uint32_t cand = __ballot_sync(0xffffffffu, jl < lim && ((s_mask[jl] >> warp) & 1u));
    while (cand) {
      const int bit = 31 - __clz(cand);
      cand ^= 1u << bit;
      const int j = c * 32 + bit;
      const float* r = s_rec + j * RS;
      const float4 r0 = *reinterpret_cast<const float4*>(r);
      const float4 r1 = *reinterpret_cast<const float4*>(r + 4);
      const float dx = fx - r0.x, dy = fy - r0.y;
      const float power = -0.5f * (r0.z * dx * dx + r1.x * dy * dy) - r0.w * dx * dy;
      const float gauss = legs_exp_neg(power);
      const float raw = r1.y * gauss;
      const float alpha = fminf(kAlphaMax, raw);
      const bool contrib = (base + j < ncon) && !(power > 0.0f) && !(alpha < kAlphaMin);
      if (!__any_sync(0xffffffffu, contrib)) continue;
      // branch-free from here on: lanes that do not contribute carry alpha = 0 (w = 0, A and T unchanged)
      const float al = contrib ? alpha : 0.f;
      const float om = 1.0f - al;
      // 1 / om for om in [0.01, 1]: MUFU.RCP + one Newton step (branch-free; __frcp_rn's range fix-up path costs 9 % of
      // the kernel)
      float rcp;
      asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rcp) : "f"(om));
      rcp = fmaf(rcp, fmaf(-om, rcp, 1.0f), rcp);
      T *= rcp;  // transmittance in front of this Gaussian
      const float w = al * T;
      float v[NV];
      float val[NC];
      const float4 r2 = *reinterpret_cast<const float4*>(r + 8);
      val[0] = r1.z; val[1] = r1.w; val[2] = r2.x; val[3] = r2.z; val[4] = r2.w;
#pragma unroll
      for (int k = 2; k < F + 1; k += 4) {
        const float4 q = *reinterpret_cast<const float4*>(r + 10 + k);
        val[3 + k] = q.x;
        if (k + 1 < F + 1) val[4 + k] = q.y;
        if (k + 2 < F + 1) val[5 + k] = q.z;
        if (k + 3 < F + 1) val[6 + k] = q.w;
      }
      float dLda = 0.f;
#pragma unroll
      for (int k = 0; k < NC; ++k) {
        v[6 + k] = w * G[k];
        if (k < NA) {
          const float d = val[k] - A[k];
          dLda = fmaf(G[k], d, dLda);
          A[k] = fmaf(al, d, A[k]);  // alpha*v + (1-alpha)*A
        }
      }
      dLda = fmaf(dLda, T, -bgG * rcp);
      // zero through the 0.99 clamp (C-15) and for lanes that do not contribute
      const float dLdg = (contrib && !(raw > kAlphaMax)) ? dLda : 0.f;
      const float dpow = raw * dLdg;
      v[0] = gauss * dLdg;
      v[1] = dpow * (r0.z * dx + r0.w * dy);
      v[2] = dpow * (r1.x * dy + r0.w * dx);
      v[3] = -0.5f * dpow * dx * dx;
      v[4] = -dpow * dx * dy;
      v[5] = -0.5f * dpow * dy * dy;
      const uint32_t g = s_idx[j];
      Bfly<NV>::reduce(v, lane);
#pragma unroll
      for (int q = 0; q < NOUT; ++q)
        if (my_base[q] && v[q] != 0.f) atomicAdd(my_base[q] + (size_t)g * my_stride[q], v[q]);
      if (my_conic && v[0] != 0.f) atomicAdd(my_conic + (size_t)g * 3, (double)v[0]);
    }
    }
  }
}

template <int F>
int launch_backward(legs_ctx* ctx, const DevCamera& dc, const legs_frame* frame, const uint32_t* vals,
                    const uint32_t* ranges, const float* out_pixels, const uint32_t* n_contrib, const float* dL,
                    int couple, const BwdOut& o, cudaStream_t st) {
  const int ntiles = dc.grid_x * dc.grid_y;
  if (couple)
    backward_kernel<F, true><<<ntiles, kTileThreads, 0, st>>>(vals, (const uint2*)ranges, frame->record, dc, out_pixels,
                                                             n_contrib, dL, o);
  else
    backward_kernel<F, false><<<ntiles, kTileThreads, 0, st>>>(vals, (const uint2*)ranges, frame->record, dc, out_pixels,
                                                              n_contrib, dL, o);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

}  // namespace

// defined in project_backward.cu
int legs_project_backward_launch(legs_ctx* ctx, const legs_gaussians* g, const DevCamera& dc, const legs_frame* frame,
                                 const double* dconic, const float* drgb, const float* dmean2d, legs_grads* grads,
                                 int accumulate, cudaStream_t st);

extern "C" {

size_t legs_backward_workspace_bytes(int64_t n, int32_t sem_dim) {
  (void)sem_dim;
  const size_t nn = (size_t)(n > 0 ? n : 1);
  return legs_align_up(nn * 3 * 8, 256) + legs_align_up(nn * 3 * 4, 256) + legs_align_up(nn * 2 * 4, 256);
}

int legs_render_backward(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam, const legs_frame* frame,
                         const uint32_t* vals_sorted, const uint32_t* ranges, const float* out_pixels,
                         const uint32_t* n_contrib, const float* dL_dpixels, int32_t flags, legs_grads* grads,
                         void* workspace, size_t workspace_bytes, void* stream) {
  if (!ctx) return LEGS_ERR_NULL;
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
  const size_t n = (size_t)g->n;
  const int F = g->sem_dim;
  const bool acc = (flags & LEGS_BWD_ACCUMULATE) != 0;
  char* ws = (char*)workspace;
  const size_t seg3d = legs_align_up(n * 3 * 8, 256), seg3 = legs_align_up(n * 3 * 4, 256);
  BwdOut o;
  o.dconic = (double*)ws;
  o.drgb = (float*)(ws + seg3d);
  // dmean2d of THIS view is needed by the projection backward, so it is reduced into scratch and added to the output
  float* dmean2d_view = (float*)(ws + seg3d + seg3);
  o.dmean2d = dmean2d_view;
  o.dopac = grads->dopacities; o.dsem = grads->dsem; o.dunc = grads->dunc;
  LEGS_CUDA_CHECK(ctx, cudaMemsetAsync(ws, 0, legs_backward_workspace_bytes(g->n, F), st));
  if (!acc) {
    LEGS_CUDA_CHECK(ctx, cudaMemsetAsync(grads->dopacities, 0, n * 4, st));
    LEGS_CUDA_CHECK(ctx, cudaMemsetAsync(grads->dsem, 0, n * F * 4, st));
    LEGS_CUDA_CHECK(ctx, cudaMemsetAsync(grads->dunc, 0, n * 4, st));
  }
  const DevCamera dc = make_dev_camera(cam);
  const int couple = (flags & LEGS_BWD_COUPLE_SEM) ? 1 : 0;
#define LEGS_BWD_CASE(FF)                                                                                            \
  case FF:                                                                                                           \
    rc = launch_backward<FF>(ctx, dc, frame, vals_sorted, ranges, out_pixels, n_contrib, dL_dpixels, couple, o, st); \
    break;
  switch (F) {
    LEGS_BWD_CASE(4) LEGS_BWD_CASE(8) LEGS_BWD_CASE(12) LEGS_BWD_CASE(16) LEGS_BWD_CASE(20) LEGS_BWD_CASE(24)
    LEGS_BWD_CASE(28) LEGS_BWD_CASE(32)
    default: return LEGS_ERR_DIM;
  }
#undef LEGS_BWD_CASE
  if (rc != LEGS_OK) return rc;
  return legs_project_backward_launch(ctx, g, dc, frame, o.dconic, o.drgb, dmean2d_view, grads, acc ? 1 : 0, st);
}

}  // extern "C"

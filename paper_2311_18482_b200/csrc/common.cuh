// common.cuh — shared host/device helpers of the legs CUDA library (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "legs.h"

struct legs_ctx {
  int device;
  int num_sms;
  int last_cuda_error;
  unsigned long long launches;
  void* encode_tiled;  // cuTensorMapEncodeTiled, resolved through the runtime (no link-time libcuda dependency)
};

#define LEGS_CUDA_CHECK(ctx, expr)                     \
  do {                                                 \
    cudaError_t e__ = (expr);                          \
    if (e__ != cudaSuccess) {                          \
      (ctx)->last_cuda_error = (int)e__;               \
      return LEGS_ERR_CUDA;                            \
    }                                                  \
  } while (0)

// Call after every kernel launch: records launch errors and counts the launch.
#define LEGS_LAUNCH_CHECK(ctx)                         \
  do {                                                 \
    cudaError_t e__ = cudaGetLastError();              \
    (ctx)->launches++;                                 \
    if (e__ != cudaSuccess) {                          \
      (ctx)->last_cuda_error = (int)e__;               \
      return LEGS_ERR_CUDA;                            \
    }                                                  \
  } while (0)

static inline bool legs_aligned16(const void* p) { return (((uintptr_t)p) & 15u) == 0; }
static inline size_t legs_align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Device-side copy of the camera (passed by value as a kernel argument).
struct DevCamera {
  int width, height, grid_x, grid_y;
  float fx, fy, cx, cy;
  float W[12];
  float near_plane;
  float bg[3];
  const unsigned int* tile_order;  // compositors only: CTA b works on tile tile_order[b] (NULL: tile b), legs_tile_order
};

static inline DevCamera make_dev_camera(const legs_camera* c) {
  DevCamera d;
  d.tile_order = nullptr;
  d.width = c->width;
  d.height = c->height;
  d.grid_x = (c->width + LEGS_TILE - 1) / LEGS_TILE;
  d.grid_y = (c->height + LEGS_TILE - 1) / LEGS_TILE;
  d.fx = c->fx; d.fy = c->fy; d.cx = c->cx; d.cy = c->cy;
  for (int i = 0; i < 12; ++i) d.W[i] = c->world_to_cam[i];
  d.near_plane = c->near_plane;
  for (int i = 0; i < 3; ++i) d.bg[i] = c->background[i];
  return d;
}

static inline int legs_check_camera(const legs_camera* c) {
  if (!c) return LEGS_ERR_NULL;
  if (c->width <= 0 || c->height <= 0 || c->width > 16384 || c->height > 16384) return LEGS_ERR_DIM;
  if (!(c->fx > 0.f) || !(c->fy > 0.f)) return LEGS_ERR_DIM;
  return LEGS_OK;
}

static inline int legs_check_gaussians(const legs_gaussians* g) {
  if (!g) return LEGS_ERR_NULL;
  if (g->n < 0 || g->n > (int64_t)0x7fffffff) return LEGS_ERR_DIM;
  if (g->sh_degree < 0 || g->sh_degree > 3) return LEGS_ERR_DIM;
  if (g->sh_coefs_stored < (g->sh_degree + 1) * (g->sh_degree + 1) || g->sh_coefs_stored > 16) return LEGS_ERR_DIM;
  if (g->sem_dim < 4 || g->sem_dim > LEGS_MAX_SEM_DIM || (g->sem_dim & 3)) return LEGS_ERR_DIM;
  if (g->n > 0) {
    if (!g->means || !g->scales || !g->quats || !g->opacities || !g->sh || !g->sem || !g->unc) return LEGS_ERR_NULL;
    if (!legs_aligned16(g->means) || !legs_aligned16(g->scales) || !legs_aligned16(g->quats) ||
        !legs_aligned16(g->opacities) || !legs_aligned16(g->sh) || !legs_aligned16(g->sem) || !legs_aligned16(g->unc))
      return LEGS_ERR_ALIGN;
  }
  return LEGS_OK;
}

static inline int legs_check_frame(const legs_frame* f) {
  if (!f) return LEGS_ERR_NULL;
  if (!f->depth || !f->radius || !f->rect || !f->mean2d || !f->conic_opacity || !f->rgb || !f->clamped ||
      !f->tiles_touched || !f->record || !f->num_instances)
    return LEGS_ERR_NULL;
  if (!legs_aligned16(f->depth) || !legs_aligned16(f->radius) || !legs_aligned16(f->rect) || !legs_aligned16(f->mean2d) ||
      !legs_aligned16(f->conic_opacity) || !legs_aligned16(f->rgb) || !legs_aligned16(f->clamped) ||
      !legs_aligned16(f->tiles_touched) || !legs_aligned16(f->record) ||
      !legs_aligned16(f->num_instances))
    return LEGS_ERR_ALIGN;
  return LEGS_OK;
}

#define LEGS_OVERFLOW_BIT (1ull << 63)

#ifdef __CUDACC__
// Thread -> pixel inside a 16x16 tile (256 threads): each warp covers an 8x4-pixel block, a compact footprint so that
// fewer warps see a small Gaussian (less divergence forward, fewer warp reductions backward).
__device__ __forceinline__ void legs_tile_pixel(int tid, int& lx, int& ly) {
  const int warp = tid >> 5, lane = tid & 31;
  lx = (lane & 7) + 8 * (warp & 1);
  ly = (lane >> 3) + 4 * (warp >> 1);
}
// Shared-memory loads through an explicit 32-bit shared-window address kept in a register: the compiler otherwise
// re-derives the window base (S2R SR_CgaCtaId + MOV + LEA) at every use inside the compositors' candidate loops.
__device__ __forceinline__ uint32_t legs_smem_addr(const void* p) {
  uint32_t a;
  asm volatile("{\n\t.reg .u64 t;\n\tcvta.to.shared.u64 t, %1;\n\tcvt.u32.u64 %0, t;\n\t}" : "=r"(a) : "l"(p));
  return a;
}
__device__ __forceinline__ float4 legs_lds128(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ uint32_t legs_lds32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ float2 legs_lds64(uint32_t addr) {
  float2 v;
  asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ ulonglong2 legs_lds128_u64(uint32_t addr) {
  ulonglong2 v;
  asm volatile("ld.shared.v2.u64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ unsigned long long legs_lds64_u64(uint32_t addr) {
  unsigned long long v;
  asm volatile("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(addr) : "memory");
  return v;
}
// exp(x) for x <= 0 as one multiply and one MUFU.EX2 (results below 2^-126 flush to zero: far under the 1/255 alpha
// threshold). Same values as __expf above that range, without its range fix-up instructions.
__device__ __forceinline__ float legs_exp_neg(float x) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x * 1.4426950408889634f));
  return r;
}
// One pixel-Gaussian pair: alpha before the 0.99 clamp, raw = o 2^-(u^2 + v^2), with (u, v) = R' (pixel - mean).
// Same value as o exp(-1/2 d^T Q d) of DESIGN.md "Forward, per pixel" (the record's R' is the scaled Cholesky factor of
// Q); q' >= 0 by construction, so the "power > 0" skip of the definition never fires here.
__device__ __forceinline__ float legs_pair_raw(float fx, float fy, const float4& r0, const float4& r1, float& u, float& v) {
  const float dx = fx - r0.x, dy = fy - r0.y;
  u = fmaf(r0.w, dy, r0.z * dx);
  v = r1.x * dy;
  const float q = fmaf(v, v, u * u);
  float g;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(g) : "f"(-q));
  return r1.y * g;
}
// Conservative culling of a Gaussian against the eight 8x4-pixel warp blocks of the tile at pixel (x0, y0): bit w is set
// unless min over block w of q'(d) = A dx^2 + 2 B dx dy + C dy^2 (d = pixel - mean) exceeds thr = log2(255 o) + margin,
// i.e. unless every pixel of the block fails the alpha >= 1/255 test. q' is convex: its minimum over the box is 0 if
// the mean lies inside, else the least of the four edge minima (1D quadratics, clamped). The tile's blocks lie on 4
// vertical and 8 horizontal lines; the unconstrained 1D minimiser and the constant term are taken once per line and
// shared by the segments on it. The fp32 rounding bound of the evaluation (one bound for the whole tile) is added to
// the threshold, so a block is never culled wrongly.
// The record holds the scaled Cholesky factor (r11, r12, r22) of the conic: q'(d) = (r11 dx + r12 dy)^2 + (r22 dy)^2 =
// A dx^2 + 2 B dx dy + C dy^2 with A = r11^2, B = r11 r12, C = r12^2 + r22^2.
__device__ __forceinline__ uint32_t legs_block_mask(float mux, float muy, float r11, float r12, float r22, float thr, int x0,
                                                    int y0) {
  if (!(thr >= 0.0f)) return 0u;
  const float A = r11 * r11, B = r11 * r12, C = fmaf(r12, r12, r22 * r22);
  float rA, rC;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rA) : "f"(A));
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rC) : "f"(C));
  const float ax = (float)x0 - mux, ay = (float)y0 - muy;
  // rounding bound: 4e-6 of the largest possible sum of the three terms' magnitudes over the tile
  const float DX = fmaxf(fabsf(ax), fabsf(ax + 15.0f)), DY = fmaxf(fabsf(ay), fabsf(ay + 15.0f));
  const float thrE = thr + 4e-6f * (A * DX * DX + C * DY * DY + 2.0f * fabsf(B) * DX * DY);
  // vertical lines dx = X: q'(v) = C v^2 + 2 B X v + A X^2, minimiser v* = -B X / C (an approximate reciprocal only moves
  // the evaluation point along the edge: the value changes by C dv^2, far inside the margin)
  float qv[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float X = ax + (float)(i == 0 ? 0 : i == 1 ? 7 : i == 2 ? 8 : 15);
    const float bx = 2.0f * B * X, cx = A * X * X, vs = -(B * X) * rC;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const float v = fminf(ay + (float)(4 * r + 3), fmaxf(ay + (float)(4 * r), vs));
      qv[i][r] = fmaf(fmaf(C, v, bx), v, cx);
    }
  }
  // horizontal lines dy = Y
  float qh[8][2];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const float Y = ay + (float)(4 * (j >> 1) + 3 * (j & 1));
    const float by = 2.0f * B * Y, cy = C * Y * Y, us = -(B * Y) * rA;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const float u = fminf(ax + (float)(8 * h + 7), fmaxf(ax + (float)(8 * h), us));
      qh[j][h] = fmaf(fmaf(A, u, by), u, cy);
    }
  }
  uint32_t m = 0;
#pragma unroll
  for (int w = 0; w < 8; ++w) {
    const int h = w & 1, r = w >> 1;
    const float bx0 = ax + (float)(8 * h), by0 = ay + (float)(4 * r);
    const bool inside = bx0 <= 0.0f && bx0 + 7.0f >= 0.0f && by0 <= 0.0f && by0 + 3.0f >= 0.0f;
    const float q = fminf(fminf(qv[2 * h][r], qv[2 * h + 1][r]), fminf(qh[2 * r][h], qh[2 * r + 1][h]));
    if (inside || !(q > thrE)) m |= 1u << w;   // also keeps the block when q is NaN
  }
  return m;
}
#endif

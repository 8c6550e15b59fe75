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
};

static inline DevCamera make_dev_camera(const legs_camera* c) {
  DevCamera d;
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
// exp(x) for x <= 0 as one multiply and one MUFU.EX2 (results below 2^-126 flush to zero: far under the 1/255 alpha
// threshold). Same values as __expf above that range, without its range fix-up instructions.
__device__ __forceinline__ float legs_exp_neg(float x) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x * 1.4426950408889634f));
  return r;
}
#endif

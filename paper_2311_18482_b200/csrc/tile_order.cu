// tile_order.cu — launch order of the compositors' CTAs: tiles with the longest lists first.
// One CTA per tile and one walk over the tile's whole list (S5 / S6, BASELINE.json north_star (3), (4)) makes the kernel's
// end the end of whichever long tile was started last. In a clustered scene (configs[4]: per-tile lists of 245 entries at the
// median, 15 068 at the maximum) row-major order left the SMs 35 % idle (ncu: sm__cycles_active 1.24 M of 1.91 M elapsed).
// Longest-first is the classic remedy (LPT list scheduling: the tail is then bounded by one short tile). An exact sort is
// not needed: tiles are bucketed by list length with four buckets per octave and laid out from the fullest bucket down.
// The order within a bucket follows the atomics (it is a schedule, not a result: outputs do not depend on it).
#include "common.cuh"

namespace {

constexpr int kOrdThreads = 1024;
constexpr int kOrdBuckets = 128;   // 32 octaves x 4

__device__ __forceinline__ int order_bucket(uint32_t count) {
  const uint32_t c = count < 0xffffffffu ? count + 1u : count;   // >= 1
  const int e = 31 - __clz(c);
  const int sub = e >= 2 ? (int)((c >> (e - 2)) & 3u) : (int)((c << (2 - e)) & 3u);
  return e * 4 + sub;   // monotone in count, 0 .. 127
}

__global__ void __launch_bounds__(kOrdThreads) tile_order_kernel(const uint2* __restrict__ ranges, int n_tiles,
                                                                 uint32_t* __restrict__ order) {
  __shared__ uint32_t s_count[kOrdBuckets];
  __shared__ uint32_t s_base[kOrdBuckets];
  for (int b = threadIdx.x; b < kOrdBuckets; b += kOrdThreads) s_count[b] = 0u;
  __syncthreads();
  for (int t = threadIdx.x; t < n_tiles; t += kOrdThreads) {
    const uint2 r = ranges[t];
    atomicAdd(&s_count[order_bucket(r.y - r.x)], 1u);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t run = 0u;
    for (int b = kOrdBuckets - 1; b >= 0; --b) { s_base[b] = run; run += s_count[b]; }
  }
  __syncthreads();
  for (int t = threadIdx.x; t < n_tiles; t += kOrdThreads) {
    const uint2 r = ranges[t];
    order[atomicAdd(&s_base[order_bucket(r.y - r.x)], 1u)] = (uint32_t)t;
  }
}

}  // namespace

extern "C" int legs_tile_order(legs_ctx* ctx, const uint32_t* ranges, int32_t n_tiles, uint32_t* tile_order, void* stream) {
  if (!ctx) return LEGS_ERR_NULL;
  if (n_tiles < 0 || n_tiles > (1 << 22)) return LEGS_ERR_DIM;
  if (n_tiles == 0) return LEGS_OK;
  if (!ranges || !tile_order) return LEGS_ERR_NULL;
  if (!legs_aligned16(ranges) || !legs_aligned16(tile_order)) return LEGS_ERR_ALIGN;
  tile_order_kernel<<<1, kOrdThreads, 0, (cudaStream_t)stream>>>((const uint2*)ranges, n_tiles, tile_order);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

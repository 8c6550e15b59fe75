// binning.cu — S2..S4: tile lists in ascending (tile, depth bits, index) order + per-tile ranges
// (BASELINE.json north_star (2); readings C-7, C-8).
//
// The defined result is that of a stable sort of 64-bit keys (tile<<32 | float_bits(depth)) emitted in index order.
// A straight LSD sort of D 12-byte pairs over 45 key bits moves ~150 B per tile instance and is the largest HBM term
// of a frame. The same permutation is reached here with ~44 B per instance:
//   1. stable radix sort of the n Gaussians by depth bits (n << D), value = index   -> order[]
//   2. inclusive prefix sum of tiles_touched[order[j]]                              -> offs[]
//   3. emission of (tile, index) pairs in depth order at offs[j]-tiles .. offs[j]   -> D pairs, already (depth, index)-sorted
//   4. stable radix sort by the ceil(log2(tiles)) tile bits only (1-2 passes)       -> (tile, depth, index) order
//   5. ranges from tile-id boundaries; optional materialisation of the 64-bit keys.
#include "common.cuh"
#include "radix_sort.cuh"

namespace {

using namespace legs_sort;

constexpr int kScanBlock = 256;
constexpr int kScanItems = 8;
constexpr int kScanTile = kScanBlock * kScanItems;  // 2048

__device__ __forceinline__ uint32_t gather_tiles(const uint32_t* order, const uint32_t* tiles, uint32_t j, uint32_t n) {
  return j < n ? tiles[order[j]] : 0u;
}

// phase 1: per-block sums of tiles_touched in depth order
__global__ void __launch_bounds__(kScanBlock) scan_sums_kernel(const uint32_t* __restrict__ order,
                                                               const uint32_t* __restrict__ tiles, uint32_t n,
                                                               unsigned long long* __restrict__ block_sums) {
  __shared__ uint32_t ws[kScanBlock / 32];
  uint32_t s = 0;
  const uint32_t base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) s += gather_tiles(order, tiles, base + k, n);
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long t = 0;
    for (int k = 0; k < kScanBlock / 32; ++k) t += ws[k];
    block_sums[blockIdx.x] = t;
  }
}

// phase 2: exclusive scan of the block sums (one CTA); checks D against the capacity
__global__ void __launch_bounds__(1024) scan_block_sums_kernel(unsigned long long* block_sums, int nb,
                                                               unsigned long long* num_instances,
                                                               unsigned long long capacity) {
  __shared__ unsigned long long warp_tot[32];
  __shared__ unsigned long long carry_s;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int base = 0; base < nb; base += 1024) {
    const int idx = base + threadIdx.x;
    const unsigned long long v = idx < nb ? block_sums[idx] : 0ull;
    unsigned long long inc = v;
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) warp_tot[wid] = inc;
    __syncthreads();
    if (wid == 0) {
      const unsigned long long w = warp_tot[lane];
      unsigned long long winc = w;
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, winc, o);
        if (lane >= o) winc += t;
      }
      warp_tot[lane] = winc - w;
    }
    __syncthreads();
    const unsigned long long excl = carry_s + warp_tot[wid] + (inc - v);
    if (idx < nb) block_sums[idx] = excl;
    __syncthreads();
    if (threadIdx.x == 1023) carry_s = excl + v;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const unsigned long long D = carry_s;
    *num_instances = D > capacity ? (D | LEGS_OVERFLOW_BIT) : D;
  }
}

// phase 3 + S3: inclusive offsets in depth order, then emission of (tile, index) pairs.
// One thread per depth-ordered Gaussian; rects with more than kSmallRect tiles are written by the whole warp.
constexpr int kSmallRect = 8;

__global__ void __launch_bounds__(kScanBlock) emit_kernel(const uint32_t* __restrict__ order,
                                                          const uint32_t* __restrict__ tiles,
                                                          const int4* __restrict__ rect,
                                                          const unsigned long long* __restrict__ block_excl,
                                                          const unsigned long long* __restrict__ num_instances,
                                                          uint32_t n, int grid_x, uint32_t* __restrict__ tkeys,
                                                          uint32_t* __restrict__ tvals) {
  __shared__ uint32_t ws[kScanBlock / 32];
  if ((*num_instances) >> 63) return;  // D > capacity: write nothing
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  // thread t of the block owns kScanItems consecutive depth-ordered Gaussians? No: to keep the emission of a warp
  // contiguous, item k of thread t is element k*256 + t of the block's 2048-element tile.
  const uint32_t tile_base = blockIdx.x * kScanTile;
  uint32_t running = (uint32_t)block_excl[blockIdx.x];
  for (int k = 0; k < kScanItems; ++k) {
    const uint32_t j = tile_base + k * kScanBlock + threadIdx.x;
    const uint32_t idx = j < n ? order[j] : 0u;
    const uint32_t cnt = j < n ? tiles[idx] : 0u;
    uint32_t inc = cnt;
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) ws[wid] = inc;
    __syncthreads();
    uint32_t pre = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kScanBlock / 32; ++w) {
      const uint32_t t = ws[w];
      if (w < wid) pre += t;
      total += t;
    }
    const uint32_t start = running + pre + inc - cnt;  // exclusive offset of this Gaussian's instances
    running += total;
    __syncthreads();
    int4 rc = make_int4(0, 0, 0, 0);
    if (cnt) rc = rect[idx];
    const int w_ = rc.z - rc.x;
    if (cnt && cnt <= (uint32_t)kSmallRect) {
      uint32_t o = start;
      for (int ty = rc.y; ty < rc.w; ++ty)
        for (int tx = rc.x; tx < rc.z; ++tx) {
          tkeys[o] = (uint32_t)(ty * grid_x + tx);
          tvals[o] = idx;
          ++o;
        }
    }
    uint32_t big = __ballot_sync(0xffffffffu, cnt > (uint32_t)kSmallRect);
    while (big) {
      const int src = __ffs(big) - 1;
      big &= big - 1;
      const uint32_t b_cnt = __shfl_sync(0xffffffffu, cnt, src);
      const uint32_t b_start = __shfl_sync(0xffffffffu, start, src);
      const uint32_t b_idx = __shfl_sync(0xffffffffu, idx, src);
      const int b_x0 = __shfl_sync(0xffffffffu, rc.x, src), b_y0 = __shfl_sync(0xffffffffu, rc.y, src);
      const int b_w = __shfl_sync(0xffffffffu, w_, src);
      for (uint32_t e = lane; e < b_cnt; e += 32) {
        const int ty = b_y0 + (int)(e / (uint32_t)b_w), tx = b_x0 + (int)(e % (uint32_t)b_w);
        tkeys[b_start + e] = (uint32_t)(ty * grid_x + tx);
        tvals[b_start + e] = b_idx;
      }
    }
  }
}

// S4b without touching the D instances: per-tile counts from the n rects through a 2D difference array
// (+1 at (x0,y0) and (x1,y1), -1 at (x1,y0) and (x0,y1); its 2D prefix sum is the number of rects covering a tile).
// Rects clamp to the image border, so a few cells are very hot: each CTA accumulates its 2048 Gaussians in a
// shared-memory copy of the array (when it fits) and adds only its nonzero cells to the global one.
constexpr int kCountItems = 8;
__global__ void __launch_bounds__(256) tile_count_kernel(const int4* __restrict__ rect, const uint32_t* __restrict__ tiles,
                                                         uint32_t n, int grid_x, int cells, int use_smem,
                                                         int* __restrict__ diff) {
  extern __shared__ int s_cnt[];
  const int pitch = grid_x + 1;
  int* d = use_smem ? s_cnt : diff;
  if (use_smem) {
    for (int i = threadIdx.x; i < cells; i += 256) s_cnt[i] = 0;
    __syncthreads();
  }
#pragma unroll
  for (int k = 0; k < kCountItems; ++k) {
    const uint32_t i = (blockIdx.x * kCountItems + k) * 256 + threadIdx.x;
    if (i < n && tiles[i] != 0) {
      const int4 r = rect[i];
      atomicAdd(&d[r.y * pitch + r.x], 1);
      atomicAdd(&d[r.y * pitch + r.z], -1);
      atomicAdd(&d[r.w * pitch + r.x], -1);
      atomicAdd(&d[r.w * pitch + r.z], 1);
    }
  }
  if (use_smem) {
    __syncthreads();
    for (int i = threadIdx.x; i < cells; i += 256) {
      const int v = s_cnt[i];
      if (v) atomicAdd(&diff[i], v);
    }
  }
}

// One CTA: 2D prefix sum of the difference array -> count per tile; exclusive scan in tile order -> ranges;
// digit histograms of the tile-id sort passes (already exclusive-scanned, as onesweep_kernel expects them).
__global__ void __launch_bounds__(1024) tile_scan_kernel(int* diff, int grid_x, int grid_y,
                                                         const unsigned long long* __restrict__ num_instances,
                                                         PassDesc pd, uint32_t* __restrict__ hist,
                                                         uint32_t* __restrict__ ranges, int use_smem) {
  __shared__ uint32_t s_hist[2 * kBins];
  __shared__ uint32_t s_warp[32];
  __shared__ uint32_t s_carry;
  const int pitch = grid_x + 1, ntiles = grid_x * grid_y;
  const bool overflow = ((*num_instances) >> 63) != 0;
  for (int i = threadIdx.x; i < 2 * kBins; i += 1024) s_hist[i] = 0;
  if (threadIdx.x == 0) s_carry = 0;
  // the array is small (6868 entries at 1600x1064): work on a shared-memory copy when it fits, else in place
  extern __shared__ int s_diff[];
  const int cells = pitch * (grid_y + 1);
  int* d = use_smem ? s_diff : diff;
  if (use_smem) {
    for (int i = threadIdx.x; i < cells; i += 1024) s_diff[i] = diff[i];
    __syncthreads();
  }
  for (int y = threadIdx.x; y < grid_y; y += 1024) {   // along x
    int run = 0;
    for (int x = 0; x < grid_x; ++x) { run += d[y * pitch + x]; d[y * pitch + x] = run; }
  }
  __syncthreads();
  for (int x = threadIdx.x; x < grid_x; x += 1024) {   // along y
    int run = 0;
    for (int y = 0; y < grid_y; ++y) { run += d[y * pitch + x]; d[y * pitch + x] = run; }
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int base = 0; base < ntiles; base += 1024) {
    const int t = base + threadIdx.x;
    const uint32_t c = t < ntiles ? (uint32_t)d[(t / grid_x) * pitch + (t % grid_x)] : 0u;
    uint32_t inc = c;
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += v;
    }
    if (lane == 31) s_warp[wid] = inc;
    __syncthreads();
    uint32_t pre = s_carry;
    for (int w = 0; w < wid; ++w) pre += s_warp[w];
    const uint32_t start = pre + inc - c;
    if (t < ntiles) {
      const bool some = c != 0 && !overflow;
      ranges[2 * t] = some ? start : 0u;
      ranges[2 * t + 1] = some ? start + c : 0u;
      if (c) {
        atomicAdd(&s_hist[((uint32_t)t >> pd.shift[0]) & ((1u << pd.bits[0]) - 1u)], c);
        if (pd.passes > 1) atomicAdd(&s_hist[kBins + (((uint32_t)t >> pd.shift[1]) & ((1u << pd.bits[1]) - 1u))], c);
      }
    }
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = start + c;
    __syncthreads();
  }
  // exclusive scan of each pass's 256 bins (warp p handles pass p)
  if (wid < pd.passes) {
    uint32_t v[8], sum = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) { v[k] = s_hist[wid * kBins + lane * 8 + k]; sum += v[k]; }
    uint32_t inc = sum;
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t u = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += u;
    }
    uint32_t run = inc - sum;
#pragma unroll
    for (int k = 0; k < 8; ++k) { hist[wid * kBins + lane * 8 + k] = run; run += v[k]; }
  }
}

// optional: 64-bit keys (tile << 32 | float_bits(depth)) in sorted order
__global__ void __launch_bounds__(256) keys64_kernel(const uint32_t* __restrict__ tkeys, const uint32_t* __restrict__ vals,
                                                     const uint32_t* __restrict__ depth_bits,
                                                     const unsigned long long* __restrict__ num_instances,
                                                     unsigned long long* __restrict__ keys64) {
  const unsigned long long v = *num_instances;
  const uint32_t D = (v >> 63) ? 0u : (uint32_t)v;
  for (uint32_t k = blockIdx.x * 256 + threadIdx.x; k < D; k += gridDim.x * 256)
    keys64[k] = ((unsigned long long)tkeys[k] << 32) | depth_bits[vals[k]];
}

struct Layout {
  size_t order_keys[2], order_vals[2], block_sums, tkeys[2], tvals, tvals2, control, control_bytes, diff, status_n, status_d, total;
  int passes_d, bits_d[2];
  uint32_t tiles_n, tiles_d;
};

Layout make_layout(int64_t n, uint64_t capacity, int width, int height) {
  Layout L;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += legs_align_up(bytes, 256); return o; };
  const size_t nn = (size_t)(n > 0 ? n : 1), cap = (size_t)(capacity > 0 ? capacity : 1);
  for (int k = 0; k < 2; ++k) { L.order_keys[k] = take(nn * 4); L.order_vals[k] = take(nn * 4); }
  L.block_sums = take(((nn + kScanTile - 1) / kScanTile + 1) * 8);
  L.tkeys[0] = take(cap * 4); L.tkeys[1] = take(cap * 4);
  L.tvals = take(cap * 4);
  L.tvals2 = take(cap * 4);
  const int gx = (width + LEGS_TILE - 1) / LEGS_TILE, gy = (height + LEGS_TILE - 1) / LEGS_TILE;
  int bits = 1;
  while ((1ll << bits) < (long long)gx * gy) ++bits;
  L.passes_d = bits <= 8 ? 1 : 2;
  L.bits_d[0] = L.passes_d == 1 ? bits : (bits + 1) / 2;
  L.bits_d[1] = bits - L.bits_d[0];
  L.tiles_n = (uint32_t)((nn + kTile - 1) / kTile);
  L.tiles_d = (uint32_t)((cap + kTile - 1) / kTile);
  // control block (zeroed once per call): 2 histogram sets, 6 tile counters, the tile difference array, look-back
  // status of all 6 passes
  L.control = off;
  const size_t hist_bytes = 2 * kMaxPasses * kBins * 4, counters = 64;
  L.diff = hist_bytes + counters;
  L.status_n = L.diff + legs_align_up((size_t)(gx + 1) * (gy + 1) * 4, 256);
  L.status_d = L.status_n + (size_t)4 * L.tiles_n * kBins * 4;
  L.control_bytes = L.status_d + (size_t)2 * L.tiles_d * kBins * 4;
  take(L.control_bytes);
  L.total = off;
  return L;
}

}  // namespace

extern "C" {

size_t legs_sort_workspace_bytes(int64_t n, uint64_t capacity, int32_t width, int32_t height) {
  return make_layout(n, capacity, width, height).total;
}

int legs_bin_and_sort(legs_ctx* ctx, const legs_frame* frame, const legs_camera* cam, int64_t n, uint64_t capacity,
                      uint64_t* keys_sorted, uint32_t* vals_sorted, uint32_t* ranges, void* workspace,
                      size_t workspace_bytes, void* stream) {
  if (!ctx) return LEGS_ERR_NULL;
  int rc;
  if ((rc = legs_check_camera(cam)) != LEGS_OK) return rc;
  if ((rc = legs_check_frame(frame)) != LEGS_OK) return rc;
  if (!vals_sorted || !ranges || !workspace) return LEGS_ERR_NULL;
  if (!legs_aligned16(vals_sorted) || !legs_aligned16(ranges) || !legs_aligned16(workspace) ||
      (keys_sorted && !legs_aligned16(keys_sorted)))
    return LEGS_ERR_ALIGN;
  if (n < 0 || n > (int64_t)0x7fffffff || capacity == 0 || capacity >= (1ull << 30)) return LEGS_ERR_DIM;
  const DevCamera dc = make_dev_camera(cam);
  if ((long long)dc.grid_x * dc.grid_y > 65536) return LEGS_ERR_DIM;
  const Layout L = make_layout(n, capacity, cam->width, cam->height);
  if (workspace_bytes < L.total) return LEGS_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  char* ws = (char*)workspace;
  const int ntiles = dc.grid_x * dc.grid_y;
  if (n == 0) {
    LEGS_CUDA_CHECK(ctx, cudaMemsetAsync(ranges, 0, (size_t)ntiles * 2 * sizeof(uint32_t), st));
    return LEGS_OK;
  }
  LEGS_CUDA_CHECK(ctx, cudaMemsetAsync(ws + L.control, 0, L.control_bytes, st));
  uint32_t* hist_n = (uint32_t*)(ws + L.control);
  uint32_t* hist_d = hist_n + kMaxPasses * kBins;
  uint32_t* counters = (uint32_t*)(ws + L.control + 2 * kMaxPasses * kBins * 4);
  uint32_t* status_n = (uint32_t*)(ws + L.control + L.status_n);
  uint32_t* status_d = (uint32_t*)(ws + L.control + L.status_d);
  uint32_t* ok[2] = {(uint32_t*)(ws + L.order_keys[0]), (uint32_t*)(ws + L.order_keys[1])};
  uint32_t* ov[2] = {(uint32_t*)(ws + L.order_vals[0]), (uint32_t*)(ws + L.order_vals[1])};
  unsigned long long* block_sums = (unsigned long long*)(ws + L.block_sums);
  uint32_t* tk[2] = {(uint32_t*)(ws + L.tkeys[0]), (uint32_t*)(ws + L.tkeys[1])};
  uint32_t* tv = (uint32_t*)(ws + L.tvals);
  uint32_t* tv2 = (uint32_t*)(ws + L.tvals2);
  const uint32_t n32 = (uint32_t)n;
  const uint32_t* depth_bits = (const uint32_t*)frame->depth;
  unsigned long long* num_inst = (unsigned long long*)frame->num_instances;

  // 1. Gaussians by depth bits: 4 x 8-bit passes, value = index
  PassDesc pn;
  pn.passes = 4;
  for (int p = 0; p < 4; ++p) { pn.shift[p] = 8 * p; pn.bits[p] = 8; }
  const int hist_grid = ctx->num_sms * 4;
  histogram_kernel<<<hist_grid, kThreads, 0, st>>>(depth_bits, nullptr, n32, pn, hist_n);
  LEGS_LAUNCH_CHECK(ctx);
  scan_histogram_kernel<<<1, 32 * kMaxPasses, 0, st>>>(hist_n, 4);
  LEGS_LAUNCH_CHECK(ctx);
  {
    const uint32_t* kin = depth_bits;
    const uint32_t* vin = nullptr;
    for (int p = 0; p < 4; ++p) {
      uint32_t* kout = p == 3 ? nullptr : ok[p & 1];
      uint32_t* vout = ov[p & 1];
      onesweep_kernel<<<L.tiles_n, kThreads, 0, st>>>(kin, vin, kout, vout, nullptr, n32, 8 * p, 8, hist_n + p * kBins,
                                                      status_n + (size_t)p * L.tiles_n * kBins, counters + p);
      LEGS_LAUNCH_CHECK(ctx);
      kin = kout; vin = vout;
    }
  }
  const uint32_t* order = ov[1];
  // 2. prefix sum of tiles_touched in depth order (block sums, then their scan; phase 3 is fused into emission)
  const int nb = (int)((n32 + kScanTile - 1) / kScanTile);
  scan_sums_kernel<<<nb, kScanBlock, 0, st>>>(order, frame->tiles_touched, n32, block_sums);
  LEGS_LAUNCH_CHECK(ctx);
  scan_block_sums_kernel<<<1, 1024, 0, st>>>(block_sums, nb, num_inst, (unsigned long long)capacity);
  LEGS_LAUNCH_CHECK(ctx);
  // 3. emission in depth order
  emit_kernel<<<nb, kScanBlock, 0, st>>>(order, frame->tiles_touched, (const int4*)frame->rect, block_sums, num_inst, n32,
                                         dc.grid_x, tk[0], tv);
  LEGS_LAUNCH_CHECK(ctx);
  // 4. stable sort by tile bits
  PassDesc pd;
  pd.passes = L.passes_d;
  pd.shift[0] = 0; pd.bits[0] = L.bits_d[0];
  pd.shift[1] = L.bits_d[0]; pd.bits[1] = L.bits_d[1];
  for (int p = 2; p < kMaxPasses; ++p) { pd.shift[p] = 0; pd.bits[p] = 1; }
  // per-tile counts from the rects -> ranges and the digit histograms of both passes (no sweep over the D instances)
  int* diff = (int*)(ws + L.control + L.diff);
  const size_t diff_bytes = (size_t)(dc.grid_x + 1) * (dc.grid_y + 1) * 4;
  const int use_smem = diff_bytes <= 40 * 1024;
  tile_count_kernel<<<(n32 + 256 * kCountItems - 1) / (256 * kCountItems), 256, use_smem ? diff_bytes : 0, st>>>(
      (const int4*)frame->rect, frame->tiles_touched, n32, dc.grid_x, (dc.grid_x + 1) * (dc.grid_y + 1), use_smem, diff);
  LEGS_LAUNCH_CHECK(ctx);
  tile_scan_kernel<<<1, 1024, use_smem ? diff_bytes : 0, st>>>(diff, dc.grid_x, dc.grid_y, num_inst, pd, hist_d, ranges,
                                                               use_smem);
  LEGS_LAUNCH_CHECK(ctx);
  const uint32_t* sorted_tiles;
  if (pd.passes == 1) {
    onesweep_kernel<<<L.tiles_d, kThreads, 0, st>>>(tk[0], tv, keys_sorted ? tk[1] : nullptr, vals_sorted, num_inst, 0, 0,
                                                    pd.bits[0], hist_d, status_d, counters + 4);
    LEGS_LAUNCH_CHECK(ctx);
    sorted_tiles = tk[1];
  } else {
    // pass 1: (tk[0], tv) -> (tk[1], tv2);  pass 2: (tk[1], tv2) -> (tk[0], vals_sorted)
    onesweep_kernel<<<L.tiles_d, kThreads, 0, st>>>(tk[0], tv, tk[1], tv2, num_inst, 0, pd.shift[0], pd.bits[0], hist_d,
                                                    status_d, counters + 4);
    LEGS_LAUNCH_CHECK(ctx);
    onesweep_kernel<<<L.tiles_d, kThreads, 0, st>>>(tk[1], tv2, keys_sorted ? tk[0] : nullptr, vals_sorted, num_inst, 0,
                                                    pd.shift[1], pd.bits[1],
                                                    hist_d + kBins, status_d + (size_t)L.tiles_d * kBins, counters + 5);
    LEGS_LAUNCH_CHECK(ctx);
    sorted_tiles = tk[0];
  }
  // 5. optional 64-bit keys
  const int sweep_grid = ctx->num_sms * 8;
  if (keys_sorted) {
    keys64_kernel<<<sweep_grid, 256, 0, st>>>(sorted_tiles, vals_sorted, depth_bits, num_inst,
                                              (unsigned long long*)keys_sorted);
    LEGS_LAUNCH_CHECK(ctx);
  }
  return LEGS_OK;
}

}  // extern "C"

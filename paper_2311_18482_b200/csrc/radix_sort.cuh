// radix_sort.cuh — hand-written stable LSD radix sort for (u32 key, u32 value) pairs, "onesweep" style:
// one up-front histogram kernel for all digit passes, then ONE kernel per digit that reads every pair once and
// writes it once (decoupled look-back across tiles instead of a separate scan + scatter).
// HBM traffic per pass: 16 B per pair (+ 1 KB of look-back state per 4096-pair tile).
//
// BASELINE.json north_star (2): "a hand-written device radix sort". Used twice by legs_bin_and_sort:
// (a) Gaussians by depth bits (n items, 4 x 8-bit passes), (b) tile instances by tile id (D items, 1-2 passes).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace legs_sort {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
#ifndef LEGS_SORT_ITEMS
#define LEGS_SORT_ITEMS 16
#endif
constexpr int kItems = LEGS_SORT_ITEMS;
constexpr int kTile = kThreads * kItems;  // 4096 pairs per CTA tile
constexpr int kBins = 256;
constexpr int kMaxPasses = 4;
constexpr uint32_t kFlagAggregate = 1u << 30;
constexpr uint32_t kFlagPrefix = 2u << 30;
constexpr uint32_t kValueMask = (1u << 30) - 1;

struct PassDesc {
  int shift[kMaxPasses];
  int bits[kMaxPasses];
  int passes;
};

// element count: host value, or device scalar (bit 63 = overflow flag -> treated as 0)
__device__ __forceinline__ uint32_t load_count(const unsigned long long* n_dev, uint32_t n_host) {
  if (!n_dev) return n_host;
  const unsigned long long v = *n_dev;
  return (v >> 63) ? 0u : (uint32_t)v;
}

// hist[pass][bin] += count of keys with that digit. Grid-stride; shared-memory privatised.
__global__ void __launch_bounds__(kThreads) histogram_kernel(const uint32_t* __restrict__ keys,
                                                             const unsigned long long* n_dev, uint32_t n_host,
                                                             PassDesc pd, uint32_t* __restrict__ hist) {
  __shared__ uint32_t sh[kMaxPasses * kBins];
  for (int i = threadIdx.x; i < kMaxPasses * kBins; i += kThreads) sh[i] = 0;
  __syncthreads();
  const uint32_t n = load_count(n_dev, n_host);
  for (uint32_t i = blockIdx.x * kThreads + threadIdx.x; i < n; i += gridDim.x * kThreads) {
    const uint32_t k = keys[i];
#pragma unroll
    for (int p = 0; p < kMaxPasses; ++p)
      if (p < pd.passes) atomicAdd(&sh[p * kBins + ((k >> pd.shift[p]) & ((1u << pd.bits[p]) - 1u))], 1u);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < pd.passes * kBins; i += kThreads)
    if (sh[i]) atomicAdd(&hist[i], sh[i]);
}

// in-place exclusive scan over the 256 bins of each pass (one block, one warp per pass)
__global__ void __launch_bounds__(32 * kMaxPasses) scan_histogram_kernel(uint32_t* hist, int passes) {
  const int p = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (p >= passes) return;
  uint32_t* h = hist + p * kBins;
  uint32_t v[8], s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) { v[k] = h[lane * 8 + k]; s += v[k]; }
  uint32_t inc = s;
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  uint32_t run = inc - s;
#pragma unroll
  for (int k = 0; k < 8; ++k) { h[lane * 8 + k] = run; run += v[k]; }
}

// One digit pass. keys_in/vals_in -> keys_out/vals_out. vals_in == nullptr means "value = index" (iota).
// keys_out may be nullptr (last pass when only the permutation is wanted).
// status: [num_tiles][256] u32, zeroed before launch; tile_counter: u32 zeroed before launch.
// global_base: histogram of this pass's digit over all elements (256 entries); base_is_scanned = 0: raw counts, every
// CTA takes their exclusive scan itself (no separate scan launch); 1: already an exclusive scan.
__global__ void __launch_bounds__(kThreads) onesweep_kernel(const uint32_t* __restrict__ keys_in,
                                                            const uint32_t* __restrict__ vals_in,
                                                            uint32_t* __restrict__ keys_out,
                                                            uint32_t* __restrict__ vals_out,
                                                            const unsigned long long* n_dev, uint32_t n_host, int shift,
                                                            int bits, const uint32_t* __restrict__ global_base,
                                                            int base_is_scanned, volatile uint32_t* status,
                                                            uint32_t* tile_counter) {
  __shared__ uint32_t s_keys[kTile];
  __shared__ uint32_t s_vals[kTile];
  __shared__ uint32_t s_warp_hist[kWarps * kBins];
  __shared__ int s_goff[kBins];        // global position of a bin's first element minus its local start
  __shared__ uint32_t s_scan[kWarps];
  __shared__ uint32_t s_tile;

  const uint32_t n = load_count(n_dev, n_host);
  if (threadIdx.x == 0) s_tile = atomicAdd(tile_counter, 1u);
  for (int i = threadIdx.x; i < kWarps * kBins; i += kThreads) s_warp_hist[i] = 0;
  __syncthreads();
  const uint32_t tile = s_tile;
  const uint32_t tile_base = tile * (uint32_t)kTile;
  if (tile_base >= n) return;
  const uint32_t n_tile = min((uint32_t)kTile, n - tile_base);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const uint32_t mask = (1u << bits) - 1u;
  // global start of bin b = exclusive scan of the digit histogram (thread b <-> bin b)
  uint32_t gbase = global_base[threadIdx.x];
  if (!base_is_scanned) {
    const uint32_t c = gbase;
    uint32_t inc = c;
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t tt = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += tt;
    }
    if (lane == 31) s_scan[wid] = inc;
    __syncthreads();
    uint32_t pre = 0;
    for (int w = 0; w < wid; ++w) pre += s_scan[w];
    gbase = pre + inc - c;
    __syncthreads();
  }

  // 1. load: warp w owns the contiguous chunk [w*512, (w+1)*512) of the tile, item i of lane l = chunk[i*32+l]
  uint32_t key[kItems], val[kItems];
  uint16_t rank[kItems];
  const uint32_t wbase = wid * (kItems * 32);
#pragma unroll
  for (int i = 0; i < kItems; ++i) {
    const uint32_t loc = wbase + i * 32 + lane;
    if (loc < n_tile) {
      key[i] = keys_in[tile_base + loc];
      val[i] = vals_in ? vals_in[tile_base + loc] : tile_base + loc;
    } else {
      key[i] = 0xffffffffu;  // padding sorts to the end of the last bin of the last tile
      val[i] = 0;
    }
  }
  // 2. per-warp stable ranking with match.any
  uint32_t* wh = s_warp_hist + wid * kBins;
#pragma unroll
  for (int i = 0; i < kItems; ++i) {
    const uint32_t d = (key[i] >> shift) & mask;
    const uint32_t peers = __match_any_sync(0xffffffffu, d);
    const uint32_t before = __popc(peers & ((1u << lane) - 1u));
    const uint32_t prev = wh[d];
    __syncwarp();
    if (before == 0) wh[d] = prev + __popc(peers);
    __syncwarp();
    rank[i] = (uint16_t)(prev + before);
  }
  __syncthreads();
  // 3. per-bin: exclusive scan over warps, tile total, look-back for the global prefix
  {
    const int b = threadIdx.x;  // kThreads == kBins
    uint32_t sum = 0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) {
      const uint32_t t = s_warp_hist[w * kBins + b];
      s_warp_hist[w * kBins + b] = sum;
      sum += t;
    }
    const uint32_t count = sum;
    volatile uint32_t* st = status + (size_t)tile * kBins + b;
    if (tile == 0) *st = kFlagPrefix | count;
    else *st = kFlagAggregate | count;
    uint32_t excl = 0;
    if (tile > 0) {
      // look-back over the predecessors' words of this bin, kLook at a time: the loads of a batch are independent (one
      // L2 round trip for the batch instead of one per predecessor); the words are then consumed in order up to the
      // first inclusive prefix, or up to a word that is not published yet (predecessor tiles hold earlier tickets, so
      // they are running), from where the next batch starts.
      constexpr int kLook = 8;
      int t = (int)tile - 1;
      bool done = false;
      while (!done) {
        uint32_t w[kLook];
#pragma unroll
        for (int k = 0; k < kLook; ++k) w[k] = t - k >= 0 ? (uint32_t)status[(size_t)(t - k) * kBins + b] : (uint32_t)(2u << 30);
        int used = 0;
#pragma unroll
        for (int k = 0; k < kLook; ++k) {
          if (!done && used == k) {
            const uint32_t f = w[k] & ~kValueMask;
            if (f != 0) {
              excl += w[k] & kValueMask;
              ++used;
              if (f == kFlagPrefix) done = true;
            }
          }
        }
        t -= used;
      }
      *st = kFlagPrefix | (excl + count);
    }
    // block-wide exclusive scan of `count` over bins -> local start of each bin
    uint32_t inc = count;
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t tt = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += tt;
    }
    if (lane == 31) s_scan[wid] = inc;
    __syncthreads();
    uint32_t pre = 0;
    for (int w = 0; w < wid; ++w) pre += s_scan[w];
    const uint32_t local_start = pre + inc - count;
    s_goff[b] = (int)(gbase + excl) - (int)local_start;
    // fold the bin's local start into every warp's offset for that bin
#pragma unroll
    for (int w = 0; w < kWarps; ++w) s_warp_hist[w * kBins + b] += local_start;
  }
  __syncthreads();
  // 4. exchange through shared memory into tile-local sorted order
#pragma unroll
  for (int i = 0; i < kItems; ++i) {
    const uint32_t d = (key[i] >> shift) & mask;
    const uint32_t pos = wh[d] + rank[i];
    s_keys[pos] = key[i];
    s_vals[pos] = val[i];
  }
  __syncthreads();
  // 5. coalesced scatter: consecutive threads hold consecutive elements of a bin run
#pragma unroll
  for (int i = 0; i < kItems; ++i) {
    const uint32_t pos = i * kThreads + threadIdx.x;
    if (pos < n_tile) {
      const uint32_t k = s_keys[pos];
      const uint32_t d = (k >> shift) & mask;
      const uint32_t g = (uint32_t)((int)pos + s_goff[d]);
      if (keys_out) keys_out[g] = k;
      vals_out[g] = s_vals[pos];
    }
  }
}

}  // namespace legs_sort

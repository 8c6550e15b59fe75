// radix_sort.cuh — hand-written stable LSD radix sort for (u32 key, u32 value) pairs, "onesweep" style:
// the digit histograms of all passes are taken up front (binning.cu: tile_count_kernel), then ONE kernel per digit reads
// every pair once and writes it once (decoupled look-back across tiles instead of a separate scan + scatter).
// HBM traffic per pass: 16 B per pair (+ 1 KB of look-back state per 4096-pair tile).
//
// BASELINE.json north_star (2): "a hand-written device radix sort". Used by legs_bin_and_sort for the Gaussians by depth
// bits (n items, 4 x 8-bit passes); the tile part of the 64-bit key never goes through a sort (binning.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace legs_sort {

#ifndef LEGS_SORT_THREADS
#define LEGS_SORT_THREADS 256
#endif
constexpr int kThreads = LEGS_SORT_THREADS;   // a multiple of 256: kSplit threads per radix bin
constexpr int kSplit = kThreads / 256;
constexpr int kWarps = kThreads / 32;
#ifndef LEGS_SORT_ITEMS
#define LEGS_SORT_ITEMS 16
#endif
constexpr int kItems = LEGS_SORT_ITEMS;
constexpr int kTile = kThreads * kItems;  // pairs per CTA tile
constexpr int kBins = 256;
constexpr int kMaxPasses = 4;
constexpr uint32_t kFlagAggregate = 1u << 30;
constexpr uint32_t kFlagPrefix = 2u << 30;
constexpr uint32_t kValueMask = (1u << 30) - 1;

// Decoupled look-back over the predecessors' status words of one column (a radix bin, or a tile row in the row-entry
// emission): publishes `count` as this tile's aggregate, sums the aggregates of the predecessors back to the nearest
// inclusive prefix, publishes the own inclusive prefix and returns the exclusive one. kLook words are loaded per round trip
// (independent loads); they are consumed in order up to the first inclusive prefix, or up to a word that is not published
// yet (predecessor tiles hold earlier tickets, so they are running), from where the next batch starts. With every tile
// of a launch resident and publishing at about the same time, tile t needs ~t / (2 kLook) round trips.
template <int kLook>
__device__ __forceinline__ uint32_t lookback(volatile uint32_t* status, uint32_t stride, uint32_t tile, uint32_t col, uint32_t count) {
  volatile uint32_t* st = status + (size_t)tile * stride + col;
  if (tile == 0) { *st = kFlagPrefix | count; return 0u; }
  *st = kFlagAggregate | count;
  uint32_t excl = 0;
  int t = (int)tile - 1;
  bool done = false;
  while (!done) {
    uint32_t w[kLook];
#pragma unroll
    for (int k = 0; k < kLook; ++k) w[k] = t - k >= 0 ? (uint32_t)status[(size_t)(t - k) * stride + col] : (uint32_t)(2u << 30);
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
  return excl;
}

// Shared memory of one digit pass (dynamic: legs_sort::kSmemBytes); a kernel that hosts a side job in one extra CTA may
// reuse it for that job.
struct SortSmem {
  uint32_t keys[kTile];
  uint32_t vals[kTile];
  uint32_t warp_hist[kWarps * kBins];
  uint32_t part[kSplit * kBins];   // per bin: totals of the kSplit groups of eight warps
  int goff[kBins];                 // global position of a bin's first element minus its local start
  uint32_t scan[8];
  uint32_t tile;
};
constexpr size_t kSmemBytes = sizeof(SortSmem);

#ifndef LEGS_SORT_LOOK
#define LEGS_SORT_LOOK 8
#endif

// One digit pass (body; kThreads threads). keys_in/vals_in -> keys_out/vals_out. vals_in == nullptr means "value =
// index" (iota). keys_out may be nullptr (last pass when only the permutation is wanted).
// status: [num_tiles][256] u32, zeroed before launch; tile_counter: u32 zeroed before launch.
// global_base: histogram of this pass's digit over all elements (256 raw counts): every CTA takes their exclusive scan
// itself (no separate scan launch).
// Tile size: the look-back is a chain over the tiles of a launch (they all run at once and publish their aggregates at
// about the same time, so tile t walks back ~t / 16 round trips before it meets an inclusive prefix); fat tiles
// (kThreads x kItems pairs) keep that chain short.
__device__ __forceinline__ void onesweep_tile(SortSmem& sm, const uint32_t* __restrict__ keys_in,
                                              const uint32_t* __restrict__ vals_in, uint32_t* __restrict__ keys_out,
                                              uint32_t* __restrict__ vals_out, uint32_t n, int shift, int bits,
                                              const uint32_t* __restrict__ global_base, volatile uint32_t* status,
                                              uint32_t* tile_counter) {
  if (threadIdx.x == 0) sm.tile = atomicAdd(tile_counter, 1u);
  for (int i = threadIdx.x; i < kWarps * kBins; i += kThreads) sm.warp_hist[i] = 0;
  __syncthreads();
  const uint32_t tile = sm.tile;
  const uint32_t tile_base = tile * (uint32_t)kTile;
  if (tile_base >= n) return;
  const uint32_t n_tile = min((uint32_t)kTile, n - tile_base);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int b = threadIdx.x & (kBins - 1), grp = threadIdx.x >> 8;   // bin and group of eight warps of this thread
  const uint32_t mask = (1u << bits) - 1u;
  // global start of bin b = exclusive scan of the digit histogram (threads of group 0: thread b <-> bin b)
  uint32_t gbase = 0, gcount = 0, ginc = 0;
  if (grp == 0) {
    gcount = global_base[b];
    ginc = gcount;
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t tt = __shfl_up_sync(0xffffffffu, ginc, o);
      if (lane >= o) ginc += tt;
    }
    if (lane == 31) sm.scan[wid] = ginc;
  }
  __syncthreads();
  if (grp == 0) {
    uint32_t pre = 0;
    for (int w = 0; w < wid; ++w) pre += sm.scan[w];
    gbase = pre + ginc - gcount;
  }
  __syncthreads();

  // 1. load: warp w owns the contiguous chunk [w*32*kItems, (w+1)*32*kItems) of the tile, item i of lane l = chunk[i*32+l]
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
  uint32_t* wh = sm.warp_hist + wid * kBins;
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
  // 3. per-bin: exclusive scan over warps (each group over its eight warps, then over the groups), tile total, look-back
  //    for the global prefix (group 0)
  {
    uint32_t sum = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
      const uint32_t t = sm.warp_hist[(grp * 8 + w) * kBins + b];
      sm.warp_hist[(grp * 8 + w) * kBins + b] = sum;
      sum += t;
    }
    if (kSplit > 1) {
      sm.part[grp * kBins + b] = sum;
      __syncthreads();
    }
    uint32_t count = 0, goffs = 0;   // tile total of the bin; entries of the bin in earlier groups
#pragma unroll
    for (int g = 0; g < kSplit; ++g) {
      const uint32_t t = kSplit > 1 ? sm.part[g * kBins + b] : sum;
      if (g < grp) goffs += t;
      count += t;
    }
    uint32_t inc = count;
    if (grp == 0) {
      const uint32_t excl = lookback<LEGS_SORT_LOOK>(status, kBins, tile, (uint32_t)b, count);
      // exclusive scan of `count` over the bins -> local start of each bin
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t tt = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += tt;
      }
      if (lane == 31) sm.scan[wid] = inc;
      gbase += excl;
    }
    __syncthreads();
    if (grp == 0) {
      uint32_t pre = 0;
      for (int w = 0; w < wid; ++w) pre += sm.scan[w];
      const uint32_t local_start = pre + inc - count;
      sm.goff[b] = (int)gbase - (int)local_start;
      if (kSplit > 1) sm.part[b] = local_start;
      goffs = local_start;
    }
    if (kSplit > 1) {
      __syncthreads();
      if (grp != 0) goffs += sm.part[b];
    }
    // fold the bin's local start (and the earlier groups' entries) into this group's warp offsets for that bin
#pragma unroll
    for (int w = 0; w < 8; ++w) sm.warp_hist[(grp * 8 + w) * kBins + b] += goffs;
  }
  __syncthreads();
  // 4. exchange through shared memory into tile-local sorted order
#pragma unroll
  for (int i = 0; i < kItems; ++i) {
    const uint32_t d = (key[i] >> shift) & mask;
    const uint32_t pos = wh[d] + rank[i];
    sm.keys[pos] = key[i];
    sm.vals[pos] = val[i];
  }
  __syncthreads();
  // 5. coalesced scatter: consecutive threads hold consecutive elements of a bin run
#pragma unroll
  for (int i = 0; i < kItems; ++i) {
    const uint32_t pos = i * kThreads + threadIdx.x;
    if (pos < n_tile) {
      const uint32_t k = sm.keys[pos];
      const uint32_t d = (k >> shift) & mask;
      const uint32_t g = (uint32_t)((int)pos + sm.goff[d]);
      if (keys_out) keys_out[g] = k;
      vals_out[g] = sm.vals[pos];
    }
  }
}

}  // namespace legs_sort

// binning.cu — S2..S4: tile lists in ascending (tile, depth bits, index) order + per-tile ranges
// (BASELINE.json north_star (2); readings C-7, C-8).
//
// The defined result is that of a stable sort of 64-bit keys (tile<<32 | float_bits(depth)) emitted in index order.
// A straight LSD sort of the D (key, value) pairs moves ~150 B per tile instance over six passes and is the largest
// HBM term of a frame. The same permutation is reached here with ONE 4-byte write per instance and no pass over D:
//   1. stable radix sort of the n Gaussians by depth bits (n << D), value = index           -> order[]
//   2. per-tile counts from a 2D difference array of the n tile rects; prefix sums           -> ranges[], D
//   3. emission, in depth order, of one entry per (Gaussian, tile ROW of its rect):
//      (row | x0 << 10 | x1 << 20, index)   (sum of rect heights ~ D / 7.5 entries)
//      straight into (row, depth) order: the position of an entry is row_start[row] + the number of earlier entries of
//      that row, a chained scan of per-row counts over blocks of depth-ordered Gaussians (no sort pass over the entries)
//   4. expansion: the row entries are cut into chunks of 1024; per chunk the number of entries covering each tile
//      column is counted, a scan over the chunks of a row gives every chunk its starting position inside each tile's
//      list, and each chunk then walks its entries in order, lane x appending values to tile (row, x)'s list.
#include "common.cuh"
#include "radix_sort.cuh"

namespace {

using namespace legs_sort;

constexpr int kScanBlock = 256;
constexpr int kScanItems = 8;
constexpr int kScanTile = kScanBlock * kScanItems;  // 2048
constexpr int kChunk = 1024;                        // row entries per expansion chunk
constexpr int kExpThreads = 128;                    // expansion CTA: one lane per tile column, 128 columns at a time
constexpr uint32_t kRowMask = 1023u;

__device__ __forceinline__ bool overflowed(const unsigned long long* num_instances) { return ((*num_instances) >> 63) != 0; }

// 32 x 32 bit-matrix transpose across the lanes of a warp: lane r holds row r (bit c = column c) on entry and column r
// (bit e = row e) on exit. Five block-swap rounds (shuffle + mask), ~30 instructions.
__device__ __forceinline__ uint32_t warp_bit_transpose(uint32_t t, int lane) {
#pragma unroll
  for (int r = 0; r < 5; ++r) {
    const int j = 16 >> r;
    const uint32_t m_lo = r == 0 ? 0x0000FFFFu : r == 1 ? 0x00FF00FFu : r == 2 ? 0x0F0F0F0Fu : r == 3 ? 0x33333333u : 0x55555555u;
    const uint32_t other = __shfl_xor_sync(0xffffffffu, t, j);
    const bool up = (lane & j) != 0;
    const uint32_t keep = up ? ~m_lo : m_lo;
    const uint32_t o = other & keep;
    t = (t & keep) | (up ? (o >> j) : (o << j));
  }
  return t;
}

// bits [lo, hi) of a 32-bit word, 0 <= lo, hi <= 32 (empty when hi <= lo)
__device__ __forceinline__ uint32_t bit_range(int lo, int hi) {
  return hi > lo ? ((hi == 32 ? 0xffffffffu : ((1u << hi) - 1u)) & ~((1u << lo) - 1u)) : 0u;
}

// Emission of the row entries straight into (row, depth) order, one pass over the depth-ordered Gaussians. A block takes a
// ticketed tile of 2048 of them; item k of thread t is element k*256 + t, so the 32 lanes of warp w at item k are 32
// consecutive Gaussians: "batch" k*8 + w, 64 batches per block, in depth order. For a batch and a group of 32 tile rows,
// lane = Gaussian builds the bit mask of the rows its rect covers, one 32 x 32 bit transpose gives lane = row the mask of
// the batch's Gaussians covering that row: its popcount is the batch's entry count of the row (pass 1), its set bits in
// ascending order are the entries in depth order (pass 2). Between the passes: per row, an exclusive scan over the 64
// batches, and the block's per-row totals go through a chained scan over the blocks (decoupled look-back, thread = row).
// Entry position = row_start[row] + entries of the row in earlier blocks + in earlier batches + its rank in the batch.
// All gathers (order -> tiles, rect) of a thread's eight items are issued before anything depends on them.
// Dynamic shared memory: base [rows_pad] u32, cnt [64][rows_pad] u16, rows_pad = grid_y rounded up to 32.
__global__ void __launch_bounds__(kScanBlock) row_emit_kernel(const uint32_t* __restrict__ order,
                                                              const uint32_t* __restrict__ tiles,
                                                              const int4* __restrict__ rect,
                                                              const unsigned long long* __restrict__ num_instances,
                                                              uint32_t n, volatile uint32_t* status, uint32_t* ticket,
                                                              const uint32_t* __restrict__ row_start, int grid_y,
                                                              uint2* __restrict__ rkv) {
  extern __shared__ uint32_t s_dyn[];
  __shared__ uint32_t s_tile;
  const int rows_pad = (grid_y + 31) & ~31, groups = rows_pad >> 5;
  uint32_t* s_base = s_dyn;
  uint16_t* s_cnt = reinterpret_cast<uint16_t*>(s_dyn + rows_pad);
  if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
  __syncthreads();
  const uint32_t tile = s_tile;
  const bool over = overflowed(num_instances);   // D > capacity: emit nothing (every block still publishes zero totals)
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const uint32_t tile_base = tile * kScanTile;
  uint32_t idx[kScanItems], tcount[kScanItems];
  uint32_t yy[kScanItems], xx[kScanItems];   // y0 | y1 << 16 (empty: 0), x0 << 10 | x1 << 20
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    const uint32_t j = tile_base + k * kScanBlock + threadIdx.x;
    idx[k] = j < n ? order[j] : 0xffffffffu;
  }
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) tcount[k] = idx[k] != 0xffffffffu ? tiles[idx[k]] : 0u;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    yy[k] = 0; xx[k] = 0;
    if (tcount[k] != 0u && !over) {
      const int4 rc = rect[idx[k]];
      yy[k] = (uint32_t)rc.y | ((uint32_t)rc.w << 16);
      xx[k] = ((uint32_t)rc.x << 10) | ((uint32_t)rc.z << 20);
    }
  }
  // pass 1: entry counts per (batch, row)
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    const int y0 = (int)(yy[k] & 0xffffu), y1 = (int)(yy[k] >> 16);
    uint16_t* crow = s_cnt + (size_t)(k * (kScanBlock / 32) + wid) * rows_pad;
    for (int g = 0; g < groups; ++g) {
      const uint32_t R = bit_range(max(y0 - 32 * g, 0), min(y1 - 32 * g, 32));
      uint32_t C = 0;
      if (__any_sync(0xffffffffu, R != 0u)) C = warp_bit_transpose(R, lane);
      crow[32 * g + lane] = (uint16_t)__popc(C);
    }
  }
  __syncthreads();
  // per row: exclusive scan over the block's batches, then the chained scan over the blocks
  for (int y = threadIdx.x; y < rows_pad; y += kScanBlock) {
    uint32_t run = 0;
    for (int b = 0; b < kScanItems * (kScanBlock / 32); ++b) {
      const uint32_t c = s_cnt[(size_t)b * rows_pad + y];
      s_cnt[(size_t)b * rows_pad + y] = (uint16_t)run;
      run += c;
    }
    const uint32_t excl = lookback<32>(status, (uint32_t)rows_pad, tile, (uint32_t)y, run);
    s_base[y] = (y < grid_y ? row_start[y] : 0u) + excl;
  }
  __syncthreads();
  // pass 2: emission, lane = row appends the batch's entries of that row in depth order
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    const int y0 = (int)(yy[k] & 0xffffu), y1 = (int)(yy[k] >> 16);
    const uint16_t* crow = s_cnt + (size_t)(k * (kScanBlock / 32) + wid) * rows_pad;
    for (int g = 0; g < groups; ++g) {
      const uint32_t R = bit_range(max(y0 - 32 * g, 0), min(y1 - 32 * g, 32));
      if (!__any_sync(0xffffffffu, R != 0u)) continue;
      uint32_t C = warp_bit_transpose(R, lane);
      const uint32_t y = (uint32_t)(32 * g + lane);
      uint32_t pos = s_base[y] + crow[y];
      const int iters = __reduce_max_sync(0xffffffffu, __popc(C));
      for (int it = 0; it < iters; ++it) {
        const int e = (__ffs(C) - 1) & 31;
        const uint32_t ve = __shfl_sync(0xffffffffu, idx[k], e);
        const uint32_t xe = __shfl_sync(0xffffffffu, xx[k], e);
        if (C) rkv[pos++] = make_uint2(y | xe, ve);
        C &= C - 1u;
      }
    }
  }
}

// Per-tile counts without touching the D instances: a 2D difference array of the n rects (+1 at (x0,y0) and (x1,y1),
// -1 at (x1,y0) and (x0,y1); its 2D prefix sum is the number of rects covering a tile). A virtual column grid_x + 1
// that every rect covers yields the number of row entries per tile row the same way. Rects clamp to the image border,
// so a few cells are very hot: each CTA accumulates its 2048 Gaussians in a shared-memory copy (when it fits) and
// adds only its nonzero cells to the global array. Pitch of the array: grid_x + 3; rows: grid_y + 1.
// The same launch also takes the four 8-bit digit histograms of the depth bits (the depth sort's global bin starts):
// both are one streaming pass over per-Gaussian arrays in index order.
constexpr int kCountItems = 8;
__global__ void __launch_bounds__(256) tile_count_kernel(const int4* __restrict__ rect, const uint32_t* __restrict__ tiles,
                                                         const uint32_t* __restrict__ depth_bits, uint32_t n, int grid_x,
                                                         int cells, int use_smem, int* __restrict__ diff,
                                                         uint32_t* __restrict__ hist) {
  extern __shared__ int s_cnt[];
  __shared__ uint32_t s_hist[4 * kBins];
  const int pitch = grid_x + 3, v = grid_x + 1;
  int* d = use_smem ? s_cnt : diff;
  for (int i = threadIdx.x; i < 4 * kBins; i += 256) s_hist[i] = 0;
  if (use_smem) {
    for (int i = threadIdx.x; i < cells; i += 256) s_cnt[i] = 0;
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < kCountItems; ++k) {
    const uint32_t i = (blockIdx.x * kCountItems + k) * 256 + threadIdx.x;
    if (i < n) {
      const uint32_t key = depth_bits[i];
#pragma unroll
      for (int p = 0; p < 4; ++p) atomicAdd(&s_hist[p * kBins + ((key >> (8 * p)) & 255u)], 1u);
    }
    if (i < n && tiles[i] != 0) {
      const int4 r = rect[i];
      atomicAdd(&d[r.y * pitch + r.x], 1);
      atomicAdd(&d[r.y * pitch + r.z], -1);
      atomicAdd(&d[r.w * pitch + r.x], -1);
      atomicAdd(&d[r.w * pitch + r.z], 1);
      atomicAdd(&d[r.y * pitch + v], 1);
      atomicAdd(&d[r.y * pitch + v + 1], -1);
      atomicAdd(&d[r.w * pitch + v], -1);
      atomicAdd(&d[r.w * pitch + v + 1], 1);
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 4 * kBins; i += 256)
    if (s_hist[i]) atomicAdd(&hist[i], s_hist[i]);
  if (use_smem) {
    for (int i = threadIdx.x; i < cells; i += 256) {
      const int c = s_cnt[i];
      if (c) atomicAdd(&diff[i], c);
    }
  }
}

// One CTA (kThreads threads): 2D prefix sum of the difference array -> count per tile and per row; exclusive scans ->
// ranges[tiles,2], row_start[grid_y + 1], *num_rows; sets bit 63 of *num_instances when D exceeds the capacity (ranges are
// then all (0,0) and *num_rows = 0). `s_mem`: shared memory for a copy of the array, used when it holds `cells` ints.
struct TileScanArgs {
  int* diff;
  int grid_x, grid_y;
  unsigned long long* num_instances;
  unsigned long long capacity;
  uint32_t* ranges;
  uint32_t* row_start;
  unsigned long long* num_rows;
};

__device__ __forceinline__ void tile_scan_body(const TileScanArgs& a, int* s_mem, int s_mem_cells, uint32_t* s_warp /*[T/32+1]*/) {
  constexpr int T = kThreads, kCarry = T / 32;
  const int grid_x = a.grid_x, grid_y = a.grid_y;
  const int pitch = grid_x + 3, ntiles = grid_x * grid_y;
  const int cells = pitch * (grid_y + 1);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const unsigned long long D64 = *a.num_instances & ~LEGS_OVERFLOW_BIT;   // the exact 64-bit sum legs_preprocess reduced
  const bool over = D64 > a.capacity;   // the 32-bit scan below wraps when D >= 2^32 and must not decide this test
  const bool use_smem = cells <= s_mem_cells;
  int* d = use_smem ? s_mem : a.diff;
  if (use_smem) {
    for (int i = threadIdx.x; i < cells; i += T) s_mem[i] = a.diff[i];
  }
  __syncthreads();
  for (int y = wid; y < grid_y; y += T / 32) {   // along x: one warp per row, 32 cells per step
    int carry = 0;
    for (int x0 = 0; x0 < pitch; x0 += 32) {
      const int x = x0 + lane;
      int v = x < pitch ? d[y * pitch + x] : 0;
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
      }
      v += carry;
      if (x < pitch) d[y * pitch + x] = v;
      carry = __shfl_sync(0xffffffffu, v, 31);
    }
  }
  __syncthreads();
  for (int x = threadIdx.x; x < pitch; x += T) {    // along y
    int run = 0;
    for (int y = 0; y < grid_y; ++y) { run += d[y * pitch + x]; d[y * pitch + x] = run; }
  }
  __syncthreads();
  if (threadIdx.x == 0) *a.num_instances = over ? (D64 | LEGS_OVERFLOW_BIT) : D64;
  // which: 0 = tiles in row-major order -> ranges, 1 = rows -> row_start
  for (int which = 0; which < 2; ++which) {
    const int count = which == 0 ? ntiles : grid_y;
    if (threadIdx.x == 0) s_warp[kCarry] = 0;   // running carry
    __syncthreads();
    for (int base = 0; base < count; base += T) {
      const int t = base + threadIdx.x;
      uint32_t c = 0;
      if (t < count) c = (uint32_t)(which == 0 ? d[(t / grid_x) * pitch + (t % grid_x)] : d[t * pitch + grid_x + 1]);
      uint32_t inc = c;
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += v;
      }
      if (lane == 31) s_warp[wid] = inc;
      __syncthreads();
      uint32_t pre = s_warp[kCarry];
      for (int w = 0; w < wid; ++w) pre += s_warp[w];
      const uint32_t start = pre + inc - c;
      if (t < count) {
        if (which == 0) {
          const bool keep = c != 0u && !over;   // D > capacity: the tile lists are not built; report empty ranges
          a.ranges[2 * t] = keep ? start : 0u;
          a.ranges[2 * t + 1] = keep ? start + c : 0u;
        } else {
          a.row_start[t] = start;
        }
      }
      __syncthreads();
      if (threadIdx.x == T - 1) s_warp[kCarry] = start + c;
      __syncthreads();
    }
    if (which == 1 && threadIdx.x == 0) {
      a.row_start[grid_y] = s_warp[kCarry];
      *a.num_rows = over ? 0ull : (unsigned long long)s_warp[kCarry];
    }
  }
}

// One 8-bit pass of the depth sort. The first pass hosts tile_scan_body in one extra CTA (the last of the grid): it
// depends only on tile_count_kernel and is on nobody's critical path until the row emission, so it costs no launch and no
// time of its own.
template <bool SIDE>
__global__ void __launch_bounds__(kThreads) depth_pass_kernel(const uint32_t* __restrict__ keys_in,
                                                              const uint32_t* __restrict__ vals_in,
                                                              uint32_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out,
                                                              uint32_t n, int shift, const uint32_t* __restrict__ hist,
                                                              volatile uint32_t* status, uint32_t* tile_counter,
                                                              TileScanArgs side) {
  extern __shared__ __align__(16) unsigned char sort_raw[];
  SortSmem& sm = *reinterpret_cast<SortSmem*>(sort_raw);
  if (SIDE && blockIdx.x == gridDim.x - 1) {
    tile_scan_body(side, reinterpret_cast<int*>(sm.keys), 2 * kTile, sm.warp_hist);   // keys + vals: 8192 contiguous ints
    return;
  }
  onesweep_tile(sm, keys_in, vals_in, keys_out, vals_out, n, shift, 8, hist, status, tile_counter);
}

// Expansion, step 1: for chunk c of the row-sorted entries, L[c][x] = number of its entries that lie in the chunk's
// LAST row and cover tile column x (what a later chunk of the same row has to skip in each tile list).
__global__ void __launch_bounds__(kExpThreads) chunk_count_kernel(const uint2* __restrict__ rkv,
                                                                  const unsigned long long* __restrict__ num_rows,
                                                                  int grid_x, int* __restrict__ L) {
  extern __shared__ int s_d[];  // grid_x + 1 difference cells
  __shared__ int s_part[kExpThreads];
  const uint32_t nr = (uint32_t)*num_rows;
  for (uint32_t chunk = blockIdx.x; chunk * (uint32_t)kChunk < nr; chunk += gridDim.x) {
    const uint32_t c0 = chunk * (uint32_t)kChunk;
    const uint32_t cn = min((uint32_t)kChunk, nr - c0);
    __syncthreads();
    for (int i = threadIdx.x; i <= grid_x; i += kExpThreads) s_d[i] = 0;
    __syncthreads();
    const uint32_t y_last = rkv[c0 + cn - 1].x & kRowMask;
    for (uint32_t i = threadIdx.x; i < cn; i += kExpThreads) {
      const uint32_t k = rkv[c0 + i].x;
      if ((k & kRowMask) == y_last) {
        atomicAdd(&s_d[(k >> 10) & 1023u], 1);
        atomicAdd(&s_d[k >> 20], -1);
      }
    }
    __syncthreads();
    // inclusive prefix over x: every thread owns a contiguous segment
    const int seg = (grid_x + kExpThreads - 1) / kExpThreads;
    const int xa = threadIdx.x * seg, xb = min(grid_x, xa + seg);
    int sum = 0;
    for (int x = xa; x < xb; ++x) sum += s_d[x];
    s_part[threadIdx.x] = sum;
    __syncthreads();
    int run = 0;
    for (int t = 0; t < (int)threadIdx.x; ++t) run += s_part[t];
    int* out = L + (size_t)chunk * grid_x;
    for (int x = xa; x < xb; ++x) { run += s_d[x]; out[x] = run; }
  }
}

// Expansion, step 2: one CTA per tile row. Cin[c][x] for every chunk c > first chunk of the row = number of the
// row's entries in earlier chunks that cover column x.
__global__ void __launch_bounds__(kExpThreads) row_carry_kernel(const uint32_t* __restrict__ row_start,
                                                                const unsigned long long* __restrict__ num_rows,
                                                                int grid_x, const int* __restrict__ L,
                                                                int* __restrict__ Cin) {
  if (*num_rows == 0) return;
  const uint32_t rs = row_start[blockIdx.x], re = row_start[blockIdx.x + 1];
  if (rs == re) return;
  const uint32_t ca = rs / kChunk, cb = (re - 1) / kChunk;
  for (int x = threadIdx.x; x < grid_x; x += kExpThreads) {
    int run = 0;
    for (uint32_t c = ca; c < cb; ++c) {
      run += L[(size_t)c * grid_x + x];   // chunk c < cb ends inside this row, so its last row is this row
      Cin[(size_t)(c + 1) * grid_x + x] = run;
    }
  }
}

// Expansion, step 3: chunks of 1024 row entries, lane <-> tile column (a warp owns a window of <= 32 columns).
// A warp compacts, with one ballot per 32 entries, the entries that overlap its columns into a ring (about a third of them
// at the benchmark's footprints) and takes them 32 at a time: lane e builds the bit mask of the warp's columns that entry
// e covers, one 32 x 32 bit transpose turns the 32 masks into "which of the 32 entries cover
// my column" per lane, and every lane appends the values of its set bits, in entry (= depth) order, to the list of tile
// (row, its column). A group whose entries span two tile rows is taken row by row.
// The append loop is warp-uniform (as many rounds as the fullest column of the group has entries): lane e keeps entry e's
// value in a register and a lane fetches the value of its next set bit with one shuffle; values go to a per-lane staging
// column in shared memory ([slot][lane]: conflict-free when the lanes are at the same slot). After each group the full
// aligned groups of four leave as 16-byte stores (every lane writes to a different list, so a 4-byte store per value would
// be one memory transaction per value); up to three values stay staged for the next group. `skip` marks the slots of the
// first group of four that lie before the list segment this chunk appends (they belong to another chunk or tile).
constexpr int kPend = 64;      // ring of pending entry indices per warp (fewer than 32 + 32 are ever pending)
constexpr int kBufSlots = 36;   // 3 carried + 32 appended per group, rounded up to a multiple of 4

template <bool KEYS>
__global__ void __launch_bounds__(kExpThreads) expand_kernel(const uint2* __restrict__ rkv,
                                                             const unsigned long long* __restrict__ num_rows,
                                                             const uint32_t* __restrict__ row_start,
                                                             const uint32_t* __restrict__ ranges, const int* __restrict__ Cin,
                                                             int grid_x, const uint32_t* __restrict__ depth_bits,
                                                             uint32_t* __restrict__ vals_sorted,
                                                             unsigned long long* __restrict__ keys_sorted) {
  __shared__ uint32_t s_k[kChunk];   // row | x0 << 10 | x1 << 20
  __shared__ uint32_t s_v[kChunk];
  __shared__ uint16_t s_pend[kExpThreads / 32][kPend];   // per warp: ring of the entries overlapping its columns, not expanded yet
  __shared__ uint32_t s_buf[kExpThreads / 32][kBufSlots][32];
  const uint32_t nr = (uint32_t)*num_rows;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t lt = (1u << lane) - 1u;
  uint32_t* buf = &s_buf[warp][0][lane];   // slot s at buf[32 * s]
  // the tile columns are cut into windows of equal width <= 32, one per warp and round (100 columns: 4 x 25, not
  // 32 + 32 + 32 + 4), so that the warps of a CTA finish a chunk together
  const int nwin = (grid_x + 31) >> 5, wcols = (grid_x + nwin - 1) / nwin;
  constexpr int kPer = kChunk / kExpThreads;   // entries per thread and chunk
  uint2 pre[kPer];                             // the next chunk, fetched while the current one is expanded
  auto fetch = [&](uint32_t chunk) {
    const uint32_t c0 = chunk * (uint32_t)kChunk;
#pragma unroll
    for (int j = 0; j < kPer; ++j) {
      const uint32_t i = c0 + j * kExpThreads + threadIdx.x;
      pre[j] = i < nr ? rkv[i] : make_uint2(0u, 0u);   // padding: x0 = x1 = 0 (covers nothing)
    }
  };
  if ((uint32_t)blockIdx.x * kChunk < nr) fetch(blockIdx.x);
  for (uint32_t chunk = blockIdx.x; chunk * (uint32_t)kChunk < nr; chunk += gridDim.x) {
    const uint32_t c0 = chunk * (uint32_t)kChunk;
    const uint32_t cn = min((uint32_t)kChunk, nr - c0);
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kPer; ++j) {
      s_k[j * kExpThreads + threadIdx.x] = pre[j].x;
      s_v[j * kExpThreads + threadIdx.x] = pre[j].y;
    }
    __syncthreads();
    if ((chunk + gridDim.x) * (unsigned long long)kChunk < nr) fetch(chunk + gridDim.x);
    const uint32_t y_first = s_k[0] & kRowMask;
    const bool continues = row_start[y_first] < c0;   // the chunk's first row began in an earlier chunk
    const uint32_t ngroups = (cn + 31u) >> 5;
    for (int wb = 0; wb < nwin; wb += kExpThreads / 32) {
      if (wb + warp >= nwin) continue;
      const int wx0 = (wb + warp) * wcols;   // this warp's first column
      const int wx1 = min(grid_x, wx0 + wcols);
      const bool col = wx0 + lane < wx1;
      const uint32_t xs = col ? (uint32_t)(wx0 + lane) : 0u;
      // ---- expansion. State of the lane's list: slot 0 of the staging column is global position `pos` (a multiple of
      // four), `cnt` slots are filled, the first `skip` of them are placeholders.
      uint32_t ycur = y_first;
      uint32_t start = ranges[2 * (ycur * grid_x + xs)] + (continues ? (uint32_t)Cin[(size_t)chunk * grid_x + xs] : 0u);
      uint32_t pos = start & ~3u, skip = start & 3u, cnt = skip;
      auto tail = [&]() {   // fewer than four slots are filled: the real ones leave as single stores
#pragma unroll
        for (uint32_t i = 0; i < 3; ++i)
          if (i >= skip && i < cnt) vals_sorted[pos + i] = buf[32 * i];
      };
      // the chunk's entries that overlap [wx0, wx1) are compacted, one ballot per 32 entries, into a small ring; whenever
      // it holds 32 (and once more at the end) a group is expanded
      uint32_t head = 0, npend = 0;
      const int wc = wx1 - wx0;
      for (uint32_t g = 0; g <= ngroups; ++g) {
        if (g < ngroups) {
          const uint32_t k = s_k[g * 32 + lane];
          const int x0 = (int)((k >> 10) & 1023u), x1 = (int)(k >> 20);
          const bool hit = x0 < wx1 && x1 > wx0;
          const uint32_t m = __ballot_sync(0xffffffffu, hit);
          if (hit) s_pend[warp][(head + npend + __popc(m & lt)) & (kPend - 1)] = (uint16_t)(g * 32 + lane);
          npend += __popc(m);
          __syncwarp();
          if (npend < 32u) continue;
        } else if (npend == 0u) {
          break;
        }
        const bool have = (uint32_t)lane < npend;
        const uint32_t qi = have ? s_pend[warp][(head + lane) & (kPend - 1)] : 0u;
        head = (head + 32u) & (kPend - 1);
        npend -= min(npend, 32u);
        const uint32_t k = have ? s_k[qi] : 0u;
        const uint32_t vmine = s_v[qi];
        const uint32_t y = k & kRowMask;
        // bits [lo, hi) of this warp's columns
        const uint32_t R = bit_range(max(0, min(wc, (int)((k >> 10) & 1023u) - wx0)), max(0, min(wc, (int)(k >> 20) - wx0)));
        uint32_t live = __ballot_sync(0xffffffffu, R != 0u);
        while (live) {   // one pass per tile row present among the group's entries (almost always one)
          const uint32_t yy = __shfl_sync(0xffffffffu, y, __ffs(live) - 1);
          const bool mine = R != 0u && y == yy;
          live &= ~__ballot_sync(0xffffffffu, mine);
          uint32_t C = warp_bit_transpose(mine ? R : 0u, lane);
          if (yy != ycur) {   // a new row starts inside the chunk: its lists start at their range begin
            tail();
            ycur = yy;
            start = ranges[2 * (yy * grid_x + xs)];
            pos = start & ~3u; skip = start & 3u; cnt = skip;
          }
          const int rounds = __reduce_max_sync(0xffffffffu, __popc(C));
          for (int it = 0; it < rounds; ++it) {
            const uint32_t v = __shfl_sync(0xffffffffu, vmine, (__ffs(C) - 1) & 31);
            if (C) {
              buf[32 * cnt] = v;
              if (KEYS) keys_sorted[pos + cnt] = ((unsigned long long)(yy * grid_x + xs) << 32) | depth_bits[v];
              ++cnt;
            }
            C &= C - 1u;
          }
          // full groups of four leave; the remainder moves to the front
          const uint32_t nfull = cnt >> 2;
          const int frounds = __reduce_max_sync(0xffffffffu, (int)nfull);
          for (int j = 0; j < frounds; ++j) {
            if ((uint32_t)j < nfull) {
              const uint4 w = make_uint4(buf[32 * (4 * j)], buf[32 * (4 * j + 1)], buf[32 * (4 * j + 2)], buf[32 * (4 * j + 3)]);
              uint32_t* dst = vals_sorted + pos + 4 * j;
              if (j == 0 && skip != 0u) {
                if (skip <= 1u) dst[1] = w.y;
                if (skip <= 2u) dst[2] = w.z;
                dst[3] = w.w;
              } else {
                *reinterpret_cast<uint4*>(dst) = w;
              }
            }
          }
          if (nfull != 0u) {
            const uint32_t t0 = buf[32 * (4 * nfull)], t1 = buf[32 * (4 * nfull + 1)], t2 = buf[32 * (4 * nfull + 2)];
            buf[0] = t0; buf[32] = t1; buf[64] = t2;
            pos += 4u * nfull; cnt &= 3u; skip = 0u;
          }
        }
      }
      tail();
      __syncwarp();
    }
  }
}

struct Layout {
  size_t order_keys[2], order_vals[2], rkv, L, Cin, row_start, control, control_bytes, diff, status_n, status_e, total;
  uint32_t emit_blocks, tiles_n, chunks;
  int rows_pad;
};

Layout make_layout(int64_t n, uint64_t capacity, int width, int height) {
  Layout L;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += legs_align_up(bytes, 256); return o; };
  const size_t nn = (size_t)(n > 0 ? n : 1), cap = (size_t)(capacity > 0 ? capacity : 1);
  const int gx = (width + LEGS_TILE - 1) / LEGS_TILE, gy = (height + LEGS_TILE - 1) / LEGS_TILE;
  for (int k = 0; k < 2; ++k) { L.order_keys[k] = take(nn * 4); L.order_vals[k] = take(nn * 4); }
  L.emit_blocks = (uint32_t)((nn + kScanTile - 1) / kScanTile);
  L.rows_pad = (gy + 31) & ~31;
  // row entries (key, value): at most one per tile instance (every rect row holds at least one tile)
  L.rkv = take(cap * 8);
  L.chunks = (uint32_t)((cap + kChunk - 1) / kChunk);
  L.L = take((size_t)L.chunks * gx * 4);
  L.Cin = take(((size_t)L.chunks + 1) * gx * 4);
  L.row_start = take((size_t)(gy + 1) * 4);
  L.tiles_n = (uint32_t)((nn + kTile - 1) / kTile);
  // control block (zeroed once per call): the four digit histograms, 4 tile counters + the emission ticket + the row-entry
  // count, the difference array, look-back status of the 4 depth passes and of the row emission
  L.control = off;
  const size_t hist_bytes = kMaxPasses * kBins * 4, counters = 64;
  L.diff = hist_bytes + counters;
  L.status_n = L.diff + legs_align_up((size_t)(gx + 3) * (gy + 1) * 4, 256);
  L.status_e = L.status_n + (size_t)4 * L.tiles_n * kBins * 4;
  L.control_bytes = L.status_e + legs_align_up((size_t)L.emit_blocks * L.rows_pad * 4, 256);
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
  // the look-back words of the sorts and scans carry 30 value bits: n and capacity stay below 2^30
  if (n < 0 || n >= (int64_t)(1ll << 30) || capacity == 0 || capacity >= (1ull << 30)) return LEGS_ERR_DIM;
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
  uint32_t* counters = (uint32_t*)(ws + L.control + kMaxPasses * kBins * 4);
  unsigned long long* num_rows = (unsigned long long*)(counters + 8);
  int* diff = (int*)(ws + L.control + L.diff);
  uint32_t* status_n = (uint32_t*)(ws + L.control + L.status_n);
  uint32_t* status_e = (uint32_t*)(ws + L.control + L.status_e);
  uint32_t* ok[2] = {(uint32_t*)(ws + L.order_keys[0]), (uint32_t*)(ws + L.order_keys[1])};
  uint32_t* ov[2] = {(uint32_t*)(ws + L.order_vals[0]), (uint32_t*)(ws + L.order_vals[1])};
  uint2* rkv = (uint2*)(ws + L.rkv);
  int* Lc = (int*)(ws + L.L);
  int* Cin = (int*)(ws + L.Cin);
  uint32_t* row_start = (uint32_t*)(ws + L.row_start);
  const uint32_t n32 = (uint32_t)n;
  const uint32_t* depth_bits = (const uint32_t*)frame->depth;
  const int4* rect = (const int4*)frame->rect;
  unsigned long long* num_inst = (unsigned long long*)frame->num_instances;

  // 1. per-tile and per-row counts from the rects (2D difference array) + the depth sort's digit histograms: one launch
  const int cells = (dc.grid_x + 3) * (dc.grid_y + 1);
  const size_t diff_bytes = (size_t)cells * 4;
  const int use_smem = diff_bytes <= 40 * 1024;
  tile_count_kernel<<<(n32 + 256 * kCountItems - 1) / (256 * kCountItems), 256, use_smem ? diff_bytes : 0, st>>>(
      rect, frame->tiles_touched, depth_bits, n32, dc.grid_x, cells, use_smem, diff, hist_n);
  LEGS_LAUNCH_CHECK(ctx);
  // 2. Gaussians by depth bits: 4 x 8-bit passes, value = index. One extra CTA of the first pass turns the difference
  //    array into ranges, row_start, the row-entry count and the overflow flag.
  if (kSmemBytes > 48 * 1024) {
    LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(depth_pass_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes));
    LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(depth_pass_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes));
  }
  TileScanArgs side;
  side.diff = diff; side.grid_x = dc.grid_x; side.grid_y = dc.grid_y;
  side.num_instances = num_inst; side.capacity = (unsigned long long)capacity;
  side.ranges = ranges; side.row_start = row_start; side.num_rows = num_rows;
  {
    const uint32_t* kin = depth_bits;
    const uint32_t* vin = nullptr;
    for (int p = 0; p < 4; ++p) {
      uint32_t* kout = p == 3 ? nullptr : ok[p & 1];
      uint32_t* vout = ov[p & 1];
      if (p == 0)
        depth_pass_kernel<true><<<L.tiles_n + 1, kThreads, kSmemBytes, st>>>(kin, vin, kout, vout, n32, 8 * p, hist_n + p * kBins,
                                                                     status_n + (size_t)p * L.tiles_n * kBins, counters + p, side);
      else
        depth_pass_kernel<false><<<L.tiles_n, kThreads, kSmemBytes, st>>>(kin, vin, kout, vout, n32, 8 * p, hist_n + p * kBins,
                                                                  status_n + (size_t)p * L.tiles_n * kBins, counters + p, side);
      LEGS_LAUNCH_CHECK(ctx);
      kin = kout; vin = vout;
    }
  }
  const uint32_t* order = ov[1];
  // 3. row entries, in (row, depth) order: ranked emission over the depth-ordered Gaussians (one launch)
  const size_t emit_smem = (size_t)L.rows_pad * 4 + (size_t)kScanItems * (kScanBlock / 32) * L.rows_pad * 2;
  if (emit_smem > 48 * 1024)
    LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(row_emit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)emit_smem));
  row_emit_kernel<<<L.emit_blocks, kScanBlock, emit_smem, st>>>(order, frame->tiles_touched, rect, num_inst, n32, status_e,
                                                                counters + 6, row_start, dc.grid_y, rkv);
  LEGS_LAUNCH_CHECK(ctx);
  // 4. expansion into the tile lists
  const size_t cc_smem = (size_t)(dc.grid_x + 1) * 4;
  const uint32_t exp_grid = L.chunks < (uint32_t)ctx->num_sms * 16u ? L.chunks : (uint32_t)ctx->num_sms * 16u;
  chunk_count_kernel<<<exp_grid, kExpThreads, cc_smem, st>>>(rkv, num_rows, dc.grid_x, Lc);
  LEGS_LAUNCH_CHECK(ctx);
  row_carry_kernel<<<dc.grid_y, kExpThreads, 0, st>>>(row_start, num_rows, dc.grid_x, Lc, Cin);
  LEGS_LAUNCH_CHECK(ctx);
  if (keys_sorted)
    expand_kernel<true><<<exp_grid, kExpThreads, 0, st>>>(rkv, num_rows, row_start, ranges, Cin, dc.grid_x, depth_bits,
                                                          vals_sorted, (unsigned long long*)keys_sorted);
  else
    expand_kernel<false><<<exp_grid, kExpThreads, 0, st>>>(rkv, num_rows, row_start, ranges, Cin, dc.grid_x, depth_bits,
                                                           vals_sorted, nullptr);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

}  // extern "C"

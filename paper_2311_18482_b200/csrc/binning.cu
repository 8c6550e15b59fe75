// binning.cu — S2..S4: tile lists in ascending (tile, depth bits, index) order + per-tile ranges
// (BASELINE.json north_star (2); readings C-7, C-8).
//
// The defined result is that of a stable sort of 64-bit keys (tile<<32 | float_bits(depth)) emitted in index order.
// A straight LSD sort of the D (key, value) pairs moves ~150 B per tile instance over six passes and is the largest
// HBM term of a frame. The same permutation is reached here with ONE 4-byte write per instance and no pass over D:
//   1. stable radix sort of the n Gaussians by depth bits (n << D), value = index           -> order[]
//   2. per-tile counts from a 2D difference array of the n tile rects; prefix sums           -> ranges[], D
//   3. emission, in depth order, of one entry per (Gaussian, tile ROW of its rect):
//      key = row | x0 << 10 | x1 << 20, value = index   (sum of rect heights ~ D / 6 entries)
//   4. stable radix sort of the row entries by the row bits only (1-2 passes)                -> per row, depth order
//   5. expansion: the row entries are cut into chunks of 1024; per chunk the number of entries covering each tile
//      column is counted, a scan over the chunks of a row gives every chunk its starting position inside each tile's
//      list, and each chunk then walks its entries in order, lane x writing value into tile (row, x)'s list.
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

// Emission of the row entries in depth order, one pass: a chained scan of the rect heights (decoupled look-back over
// ticketed blocks of 2048 depth-ordered Gaussians, as in the radix sort) fused with the emission itself. Item k of thread
// t is element k*256 + t of the block's tile, so that a warp's entries are contiguous. All gathers (order -> tiles, rect)
// of a thread's eight items are issued before anything depends on them. The last block writes the total to *num_rows
// (0 if D exceeded the capacity: nothing is emitted then).
__global__ void __launch_bounds__(kScanBlock) row_emit_kernel(const uint32_t* __restrict__ order,
                                                              const uint32_t* __restrict__ tiles,
                                                              const int4* __restrict__ rect,
                                                              const unsigned long long* __restrict__ num_instances,
                                                              uint32_t n, uint32_t nblocks, volatile uint32_t* status,
                                                              uint32_t* ticket, unsigned long long* __restrict__ num_rows,
                                                              uint32_t* __restrict__ rkeys, uint32_t* __restrict__ rvals) {
  __shared__ uint32_t ws[kScanBlock / 32];
  __shared__ uint32_t s_tile, s_prefix;
  if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
  __syncthreads();
  const uint32_t tile = s_tile;
  const bool over = overflowed(num_instances);   // D > capacity: write nothing (every block still publishes a zero total)
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const uint32_t tile_base = tile * kScanTile;
  uint32_t idx[kScanItems], cnt[kScanItems];
  int4 rc[kScanItems];
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    const uint32_t j = tile_base + k * kScanBlock + threadIdx.x;
    idx[k] = j < n ? order[j] : 0xffffffffu;
  }
  uint32_t tcount[kScanItems];
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) tcount[k] = idx[k] != 0xffffffffu ? tiles[idx[k]] : 0u;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    rc[k] = make_int4(0, 0, 0, 0);
    cnt[k] = 0;
    if (tcount[k] != 0u && !over) { rc[k] = rect[idx[k]]; cnt[k] = (uint32_t)(rc[k].w - rc[k].y); }
  }
  // block total -> published at once, then the look-back for this block's exclusive prefix
  uint32_t tsum = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) tsum += cnt[k];
  for (int o = 16; o > 0; o >>= 1) tsum += __shfl_xor_sync(0xffffffffu, tsum, o);
  if (lane == 0) ws[wid] = tsum;
  __syncthreads();
  if (wid == 0) {
    // one warp: block total, publication, and a warp-wide look-back (lane l reads the word of predecessor l of the
    // current window: 32 independent loads per round trip)
    uint32_t total = lane < kScanBlock / 32 ? ws[lane] : 0u;
    for (int o = 16; o > 0; o >>= 1) total += __shfl_xor_sync(0xffffffffu, total, o);
    uint32_t excl = 0;
    if (tile == 0) {
      if (lane == 0) status[0] = kFlagPrefix | total;
    } else {
      if (lane == 0) status[tile] = kFlagAggregate | total;
      int t = (int)tile - 1;   // nearest predecessor of the current window
      while (true) {
        const int mine = t - lane;
        const uint32_t sv = mine >= 0 ? (uint32_t)status[mine] : (uint32_t)(2u << 30);
        const uint32_t f = sv & ~kValueMask;
        const uint32_t unpub = __ballot_sync(0xffffffffu, f == 0);
        const uint32_t pref = __ballot_sync(0xffffffffu, f == kFlagPrefix);
        // usable lanes: those before the first unpublished word; stop at the first inclusive prefix among them
        const int first_unpub = unpub ? __ffs(unpub) - 1 : 32;
        const int first_pref = pref ? __ffs(pref) - 1 : 32;
        const int upto = first_pref < first_unpub ? first_pref + 1 : first_unpub;   // lanes [0, upto) are consumed
        uint32_t v = lane < upto ? (sv & kValueMask) : 0u;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        excl += v;
        if (first_pref < first_unpub) break;
        t -= upto;   // predecessors hold earlier tickets, so they are running: the unpublished word is read again
      }
      if (lane == 0) status[tile] = kFlagPrefix | (excl + total);
    }
    if (lane == 0) {
      s_prefix = excl;
      if (tile == nblocks - 1) *num_rows = over ? 0ull : (unsigned long long)(excl + total);
    }
  }
  __syncthreads();
  uint32_t running = s_prefix;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    uint32_t inc = cnt[k];
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    __syncthreads();
    if (lane == 31) ws[wid] = inc;
    __syncthreads();
    uint32_t pre = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kScanBlock / 32; ++w) {
      const uint32_t t = ws[w];
      if (w < wid) pre += t;
      total += t;
    }
    uint32_t o = running + pre + inc - cnt[k];  // exclusive offset of this Gaussian's row entries
    running += total;
    const uint32_t xx = ((uint32_t)rc[k].x << 10) | ((uint32_t)rc[k].z << 20);
    for (int y = rc[k].y; y < rc[k].w; ++y, ++o) {
      rkeys[o] = (uint32_t)y | xx;
      rvals[o] = idx[k];
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

// One CTA: 2D prefix sum of the difference array -> count per tile and per row; exclusive scans -> ranges[tiles,2],
// row_start[grid_y + 1]; sets bit 63 of *num_instances when D exceeds the capacity (ranges are then all (0,0)).
__global__ void __launch_bounds__(1024) tile_scan_kernel(int* diff, int grid_x, int grid_y,
                                                         unsigned long long* num_instances, unsigned long long capacity,
                                                         uint32_t* __restrict__ ranges, uint32_t* __restrict__ row_start,
                                                         int use_smem) {
  extern __shared__ int s_diff[];
  __shared__ uint32_t s_warp[32];
  __shared__ uint32_t s_carry;
  const int pitch = grid_x + 3, ntiles = grid_x * grid_y;
  const int cells = pitch * (grid_y + 1);
  const unsigned long long D64 = *num_instances & ~LEGS_OVERFLOW_BIT;   // read before anything below rewrites it
  int* d = use_smem ? s_diff : diff;
  if (use_smem) {
    for (int i = threadIdx.x; i < cells; i += 1024) s_diff[i] = diff[i];
  }
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  for (int y = threadIdx.x; y < grid_y; y += 1024) {   // along x
    int run = 0;
    for (int x = 0; x < pitch; ++x) { run += d[y * pitch + x]; d[y * pitch + x] = run; }
  }
  __syncthreads();
  for (int x = threadIdx.x; x < pitch; x += 1024) {    // along y
    int run = 0;
    for (int y = 0; y < grid_y; ++y) { run += d[y * pitch + x]; d[y * pitch + x] = run; }
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  // which: 0 = tiles in row-major order -> ranges (and D), 1 = rows -> row_start
  for (int which = 0; which < 2; ++which) {
    const int count = which == 0 ? ntiles : grid_y;
    bool over = false;
    if (which == 1) {   // flag the overflow before anything is written from the scan
      // D is taken from the exact 64-bit sum legs_preprocess reduced into *num_instances: the 32-bit scan above wraps when
      // D >= 2^32 (tens of thousands of screen-filling Gaussians) and must not decide this test
      const unsigned long long D = D64;
      over = D > capacity;
      __syncthreads();
      if (threadIdx.x == 0) { *num_instances = over ? (D | LEGS_OVERFLOW_BIT) : D; s_carry = 0; }
      __syncthreads();
    }
    for (int base = 0; base < count; base += 1024) {
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
      uint32_t pre = s_carry;
      for (int w = 0; w < wid; ++w) pre += s_warp[w];
      const uint32_t start = pre + inc - c;
      if (t < count) {
        if (which == 0) { ranges[2 * t] = c ? start : 0u; ranges[2 * t + 1] = c ? start + c : 0u; }
        else row_start[t] = start;
      }
      __syncthreads();
      if (threadIdx.x == 1023) s_carry = start + c;
      __syncthreads();
    }
    if (which == 1) {   // total at [grid_y]; the unused bins up to 256 too (the one-pass row sort reads 256 bins)
      for (int t = grid_y + (int)threadIdx.x; t <= (grid_y > 256 ? grid_y : 256); t += 1024) row_start[t] = s_carry;
    }
    if (which == 1 && over) {   // D > capacity: the tile lists are not built; report empty ranges
      for (int t = threadIdx.x; t < ntiles; t += 1024) { ranges[2 * t] = 0u; ranges[2 * t + 1] = 0u; }
    }
  }
}

// Expansion, step 1: for chunk c of the row-sorted entries, L[c][x] = number of its entries that lie in the chunk's
// LAST row and cover tile column x (what a later chunk of the same row has to skip in each tile list).
__global__ void __launch_bounds__(kExpThreads) chunk_count_kernel(const uint32_t* __restrict__ rkeys,
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
    const uint32_t y_last = rkeys[c0 + cn - 1] & kRowMask;
    for (uint32_t i = threadIdx.x; i < cn; i += kExpThreads) {
      const uint32_t k = rkeys[c0 + i];
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

// Expansion, step 3: chunks of 1024 row entries, lane <-> tile column (a warp owns 32 columns, a CTA 128 at a time).
// A warp first compacts, with one ballot per 32 entries, the entries that overlap its 32 columns into a queue (about a
// third of them at the benchmark's footprints). The queue is then taken 32 at a time: lane e builds the bit mask of the
// warp's columns that entry e covers, one 32 x 32 bit transpose turns the 32 masks into "which of the 32 entries cover
// my column" per lane, and every lane appends the values of its set bits, in entry (= depth) order, to the list of tile
// (row, its column). A group whose entries span two tile rows is taken row by row. Appends go through a 4-value shift
// register and leave as one 16-byte store per aligned group of four (every lane writes to a different list, so a 4-byte
// store per value would cost one memory transaction per value). Grid-stride over the chunks.
template <bool KEYS>
__global__ void __launch_bounds__(kExpThreads) expand_kernel(const uint32_t* __restrict__ rkeys,
                                                             const uint32_t* __restrict__ rvals,
                                                             const unsigned long long* __restrict__ num_rows,
                                                             const uint32_t* __restrict__ row_start,
                                                             const uint32_t* __restrict__ ranges, const int* __restrict__ Cin,
                                                             int grid_x, const uint32_t* __restrict__ depth_bits,
                                                             uint32_t* __restrict__ vals_sorted,
                                                             unsigned long long* __restrict__ keys_sorted) {
  __shared__ uint32_t s_k[kChunk];   // row | x0 << 10 | x1 << 20
  __shared__ uint32_t s_v[kChunk];
  __shared__ uint16_t s_q[kExpThreads / 32][kChunk];   // per warp: indices of the entries overlapping its columns
  const uint32_t nr = (uint32_t)*num_rows;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t lt = (1u << lane) - 1u;
  for (uint32_t chunk = blockIdx.x; chunk * (uint32_t)kChunk < nr; chunk += gridDim.x) {
    const uint32_t c0 = chunk * (uint32_t)kChunk;
    const uint32_t cn = min((uint32_t)kChunk, nr - c0);
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < (uint32_t)kChunk; i += kExpThreads) {
      s_k[i] = i < cn ? rkeys[c0 + i] : 0u;   // padding: x0 = x1 = 0 (covers nothing)
      s_v[i] = i < cn ? rvals[c0 + i] : 0u;
    }
    __syncthreads();
    const uint32_t y_first = s_k[0] & kRowMask;
    const bool continues = row_start[y_first] < c0;   // the chunk's first row began in an earlier chunk
    const uint32_t ngroups = (cn + 31u) >> 5;
    for (int xb = 0; xb < grid_x; xb += kExpThreads) {
      const int wx0 = xb + 32 * warp;   // this warp's first column
      if (wx0 >= grid_x) continue;
      const bool col = wx0 + lane < grid_x;
      const uint32_t xs = col ? (uint32_t)(wx0 + lane) : 0u;
      // ---- compaction of the entries that overlap [wx0, wx0 + 32)
      uint32_t nq = 0;
      for (uint32_t g = 0; g < ngroups; ++g) {
        const uint32_t k = s_k[g * 32 + lane];
        const int x0 = (int)((k >> 10) & 1023u), x1 = (int)(k >> 20);
        const bool hit = x0 < wx0 + 32 && x1 > wx0;
        const uint32_t m = __ballot_sync(0xffffffffu, hit);
        if (hit) s_q[warp][nq + __popc(m & lt)] = (uint16_t)(g * 32 + lane);
        nq += __popc(m);
      }
      __syncwarp();
      // ---- expansion
      uint32_t ycur = y_first;
      uint32_t pos = ranges[2 * (ycur * grid_x + xs)] + (continues ? (uint32_t)Cin[(size_t)chunk * grid_x + xs] : 0u);
      // shift register of the last four appended values; nb of them are not written yet. Invariant: (pos - nb) % 4 == 0
      // or nb < 4 values sit at the unaligned head of the segment this chunk appends.
      uint32_t b0 = 0, b1 = 0, b2 = 0, b3 = 0, nb = 0;
      auto flush = [&]() {   // the nb pending values are the last nb of (b0..b3), at positions pos - nb .. pos - 1
        if (nb >= 3) vals_sorted[pos - 3] = b1;
        if (nb >= 2) vals_sorted[pos - 2] = b2;
        if (nb >= 1) vals_sorted[pos - 1] = b3;
        nb = 0;
      };
      for (uint32_t q0 = 0; q0 < nq; q0 += 32) {
        const bool have = q0 + lane < nq;
        const uint32_t k = have ? s_k[s_q[warp][q0 + lane]] : 0u;
        const uint32_t y = k & kRowMask;
        const int lo = max(0, min(32, (int)((k >> 10) & 1023u) - wx0)), hi = max(0, min(32, (int)(k >> 20) - wx0));
        // bits [lo, hi) of this warp's columns
        const uint32_t R = hi > lo ? ((hi == 32 ? 0xffffffffu : ((1u << hi) - 1u)) & ~((1u << lo) - 1u)) : 0u;
        uint32_t live = __ballot_sync(0xffffffffu, R != 0u);
        while (live) {   // one pass per tile row present among the group's entries (almost always one)
          const uint32_t yy = __shfl_sync(0xffffffffu, y, __ffs(live) - 1);
          const bool mine = R != 0u && y == yy;
          live &= ~__ballot_sync(0xffffffffu, mine);
          uint32_t C = warp_bit_transpose(mine ? R : 0u, lane);
          if (yy != ycur) {   // a new row starts inside the chunk: its lists start at their range begin
            flush();
            ycur = yy;
            pos = ranges[2 * (yy * grid_x + xs)];
          }
          while (C) {
            const uint32_t e = (uint32_t)__ffs(C) - 1u;
            C &= C - 1u;
            const uint32_t v = s_v[s_q[warp][q0 + e]];
            if (KEYS) keys_sorted[pos] = ((unsigned long long)(yy * grid_x + xs) << 32) | depth_bits[v];
            b0 = b1; b1 = b2; b2 = b3; b3 = v;
            ++pos; ++nb;
            if ((pos & 3u) == 0u) {   // an aligned group of four ends here
              if (nb >= 4) *reinterpret_cast<uint4*>(vals_sorted + pos - 4) = make_uint4(b0, b1, b2, b3);
              else flush();           // the unaligned head of the segment (fewer than four values)
              nb = 0;
            }
          }
        }
      }
      flush();
      __syncwarp();
    }
  }
}

struct Layout {
  size_t order_keys[2], order_vals[2], rkeys[2], rvals[2], L, Cin, row_start, control, control_bytes, diff,
      status_n, status_r, status_e, total;
  uint32_t emit_blocks;
  int passes_r, bits_r[2];
  uint32_t tiles_n, tiles_r, chunks;
};

Layout make_layout(int64_t n, uint64_t capacity, int width, int height) {
  Layout L;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += legs_align_up(bytes, 256); return o; };
  const size_t nn = (size_t)(n > 0 ? n : 1), cap = (size_t)(capacity > 0 ? capacity : 1);
  const int gx = (width + LEGS_TILE - 1) / LEGS_TILE, gy = (height + LEGS_TILE - 1) / LEGS_TILE;
  for (int k = 0; k < 2; ++k) { L.order_keys[k] = take(nn * 4); L.order_vals[k] = take(nn * 4); }
  L.emit_blocks = (uint32_t)((nn + kScanTile - 1) / kScanTile);
  // row entries: at most one per tile instance (every rect row holds at least one tile)
  for (int k = 0; k < 2; ++k) { L.rkeys[k] = take(cap * 4); L.rvals[k] = take(cap * 4); }
  L.chunks = (uint32_t)((cap + kChunk - 1) / kChunk);
  L.L = take((size_t)L.chunks * gx * 4);
  L.Cin = take(((size_t)L.chunks + 1) * gx * 4);
  L.row_start = take((size_t)(gy + 1 > 257 ? gy + 1 : 257) * 4);   // >= 257 entries: read as a 256-bin scan by the row sort
  int bits = 1;
  while ((1 << bits) < gy) ++bits;
  L.passes_r = bits <= 8 ? 1 : 2;
  L.bits_r[0] = L.passes_r == 1 ? bits : (bits + 1) / 2;
  L.bits_r[1] = bits - L.bits_r[0];
  L.tiles_n = (uint32_t)((nn + kTile - 1) / kTile);
  L.tiles_r = (uint32_t)((cap + kTile - 1) / kTile);
  // control block (zeroed once per call): 2 histogram sets, 6 tile counters + the row-entry count, the difference
  // array, look-back status of all 6 passes
  L.control = off;
  const size_t hist_bytes = 2 * kMaxPasses * kBins * 4, counters = 64;
  L.diff = hist_bytes + counters;
  L.status_n = L.diff + legs_align_up((size_t)(gx + 3) * (gy + 1) * 4, 256);
  L.status_r = L.status_n + (size_t)4 * L.tiles_n * kBins * 4;
  L.status_e = L.status_r + (size_t)2 * L.tiles_r * kBins * 4;
  L.control_bytes = L.status_e + legs_align_up((size_t)L.emit_blocks * 4, 256);
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
  uint32_t* hist_r = hist_n + kMaxPasses * kBins;
  uint32_t* counters = (uint32_t*)(ws + L.control + 2 * kMaxPasses * kBins * 4);
  unsigned long long* num_rows = (unsigned long long*)(counters + 8);
  int* diff = (int*)(ws + L.control + L.diff);
  uint32_t* status_n = (uint32_t*)(ws + L.control + L.status_n);
  uint32_t* status_r = (uint32_t*)(ws + L.control + L.status_r);
  uint32_t* ok[2] = {(uint32_t*)(ws + L.order_keys[0]), (uint32_t*)(ws + L.order_keys[1])};
  uint32_t* ov[2] = {(uint32_t*)(ws + L.order_vals[0]), (uint32_t*)(ws + L.order_vals[1])};
  uint32_t* status_e = (uint32_t*)(ws + L.control + L.status_e);
  uint32_t* rk[2] = {(uint32_t*)(ws + L.rkeys[0]), (uint32_t*)(ws + L.rkeys[1])};
  uint32_t* rv[2] = {(uint32_t*)(ws + L.rvals[0]), (uint32_t*)(ws + L.rvals[1])};
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
  // 2. Gaussians by depth bits: 4 x 8-bit passes, value = index
  {
    const uint32_t* kin = depth_bits;
    const uint32_t* vin = nullptr;
    for (int p = 0; p < 4; ++p) {
      uint32_t* kout = p == 3 ? nullptr : ok[p & 1];
      uint32_t* vout = ov[p & 1];
      onesweep_kernel<<<L.tiles_n, kThreads, 0, st>>>(kin, vin, kout, vout, nullptr, n32, 8 * p, 8, hist_n + p * kBins, 0,
                                                      status_n + (size_t)p * L.tiles_n * kBins, counters + p);
      LEGS_LAUNCH_CHECK(ctx);
      kin = kout; vin = vout;
    }
  }
  const uint32_t* order = ov[1];
  // ranges, row_start, D (+ overflow flag) from the difference array
  tile_scan_kernel<<<1, 1024, use_smem ? diff_bytes : 0, st>>>(diff, dc.grid_x, dc.grid_y, num_inst,
                                                               (unsigned long long)capacity, ranges, row_start, use_smem);
  LEGS_LAUNCH_CHECK(ctx);
  // 3. row entries in depth order: chained scan of the rect heights fused with the emission (one launch)
  row_emit_kernel<<<L.emit_blocks, kScanBlock, 0, st>>>(order, frame->tiles_touched, rect, num_inst, n32, L.emit_blocks, status_e,
                                                        counters + 6, num_rows, rk[0], rv[0]);
  LEGS_LAUNCH_CHECK(ctx);
  // 4. stable sort of the row entries by their row bits
  PassDesc pr;
  pr.passes = L.passes_r;
  pr.shift[0] = 0; pr.bits[0] = L.bits_r[0];
  pr.shift[1] = L.bits_r[0]; pr.bits[1] = L.bits_r[1] > 0 ? L.bits_r[1] : 1;
  for (int p = 2; p < kMaxPasses; ++p) { pr.shift[p] = 0; pr.bits[p] = 1; }
  // one pass (at most 256 tile rows): the digit is the row, whose exclusive scan tile_scan_kernel already wrote
  // (row_start, padded to 257 entries); two passes: the generic histogram of both digits
  if (pr.passes > 1) {
    histogram_kernel<<<ctx->num_sms * 4, kThreads, 0, st>>>(rk[0], num_rows, 0, pr, hist_r);
    LEGS_LAUNCH_CHECK(ctx);
  }
  int cur = 0;
  for (int p = 0; p < pr.passes; ++p) {
    const bool scanned = pr.passes == 1;
    onesweep_kernel<<<L.tiles_r, kThreads, 0, st>>>(rk[cur], rv[cur], rk[cur ^ 1], rv[cur ^ 1], num_rows, 0, pr.shift[p],
                                                    pr.bits[p], scanned ? row_start : hist_r + p * kBins, scanned ? 1 : 0,
                                                    status_r + (size_t)p * L.tiles_r * kBins, counters + 4 + p);
    LEGS_LAUNCH_CHECK(ctx);
    cur ^= 1;
  }
  // 5. expansion into the tile lists
  const size_t cc_smem = (size_t)(dc.grid_x + 1) * 4;
  const uint32_t exp_grid = L.chunks < (uint32_t)ctx->num_sms * 16u ? L.chunks : (uint32_t)ctx->num_sms * 16u;
  chunk_count_kernel<<<exp_grid, kExpThreads, cc_smem, st>>>(rk[cur], num_rows, dc.grid_x, Lc);
  LEGS_LAUNCH_CHECK(ctx);
  row_carry_kernel<<<dc.grid_y, kExpThreads, 0, st>>>(row_start, num_rows, dc.grid_x, Lc, Cin);
  LEGS_LAUNCH_CHECK(ctx);
  if (keys_sorted)
    expand_kernel<true><<<exp_grid, kExpThreads, 0, st>>>(rk[cur], rv[cur], num_rows, row_start, ranges, Cin, dc.grid_x,
                                                          depth_bits, vals_sorted, (unsigned long long*)keys_sorted);
  else
    expand_kernel<false><<<exp_grid, kExpThreads, 0, st>>>(rk[cur], rv[cur], num_rows, row_start, ranges, Cin, dc.grid_x,
                                                           depth_bits, vals_sorted, nullptr);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

}  // extern "C"

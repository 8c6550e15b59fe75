// decode.cu — S9 + S10: per-pixel codebook decode (PAPER.md:118-122 Eq. 8; :333-358 Eq. 21-22, Table 3):
//   probs = softmax(D_MLP(x)),  decoded = probs . S          x: [P, in] bf16, S: [K, d] bf16
// and S11 relevancy (reading C-21).
//
// This step is a dense contraction, so it runs on the 5th-generation tensor cores: tcgen05.mma with fp32
// accumulators in TMEM, operands in shared memory in the K-major 128-byte-swizzled layout, weight/codebook tiles
// streamed by bulk async copies (TMA engine, mbarrier completion) through a 6-stage ring. One persistent CTA per SM;
// tile = 128 pixels (= the 128 TMEM lanes). Warp roles: warp 0 = copy producer, warp 1 = MMA issuer (one elected
// lane) + TMEM allocation, warps 2-5 = 128 row threads (first layer on the FP32 pipes, bias/ReLU, softmax,
// bf16 conversion and stores).
//
// The first MLP layer (in_dim = 8 or 16) is < 1% of the MACs and is evaluated by the row threads directly from the
// global feature row; every other layer and the probs x codebook product are UMMAs.
#include <cuda.h>
#include <string.h>

#include <algorithm>
#include <mutex>

#include "common.cuh"
#include "tc05.cuh"
#include "tmap.cuh"

namespace {

using namespace tc05;

constexpr int kRows = 128;             // pixels per tile = TMEM lanes
constexpr int kUnitBytes = 16384;      // one B unit: [128 n][64 k] bf16, SW128 K-major
constexpr int kFrontWarps = 8;
constexpr int kThreads = 32 * (2 + kFrontWarps + 8);  // warp 0 producer, warp 1 MMA issuer, warps 2-9 front group, warps 10-17 epilogue group
constexpr int kMaxHidden = 256;
constexpr int kTmemCols = 512;
constexpr int kColAp = 128;            // with hidden/logits <= 128 columns: probabilities (packed bf16 A operand) at [128,256), 64 per buffer
constexpr int kColDecode = 256;        // TMEM columns: [0,256) hidden / logits accumulators, [256,512) two decode buffers

struct DecodeParams {
  long long P;
  int n_layers;           // 2 or 3
  int dims[4];            // in, h0, (h1,) K
  int d;                  // codebook width
  int mlp_units;          // B units of the UMMA MLP layers, per tile
  int dec_units;          // B units of the codebook, per tile (0 if decoded == NULL)
  const uint16_t* feat;
  const uint8_t* units;   // packed B units (workspace)
  const float* consts;    // fp32: W0 [h0][in], then biases of layer 0,1,(2) (zeros when absent)
  uint16_t* probs;
  uint16_t* decoded;
  long long num_tiles;
};

// ---------------------------------------------------------------------------------------------------------
// pack kernel: weights/codebook -> B units in consumption order; first layer + biases -> fp32 constants
struct PackParams {
  int n_layers, dims[4], d;
  const uint16_t* w[3];
  const float* b[3];
  const uint16_t* codebook;
  uint8_t* units;
  float* consts;
  int mlp_units, dec_units;
};

__device__ __forceinline__ float bf16_to_f32(uint16_t v) { return __uint_as_float((uint32_t)v << 16); }

__global__ void __launch_bounds__(256) pack_kernel(PackParams p) {
  const int total_units = p.mlp_units + p.dec_units;
  const int tid = blockIdx.x * blockDim.x + threadIdx.x, nthreads = gridDim.x * blockDim.x;
  // B units: one thread per 16-byte chunk (8 bf16 along k)
  for (int c = tid; c < total_units * (kUnitBytes / 16); c += nthreads) {
    const int u = c / (kUnitBytes / 16), w = c % (kUnitBytes / 16);
    const int r = w / 8, ch = w % 8;  // row within the unit, 16-byte chunk within the 128-byte row
    // which matrix, which (n-chunk, k-block)?
    int uu = u, rows = 0, cols = 0, nc = 0, kb = 0;
    const uint16_t* src = nullptr;
    bool transposed = false;
    if (u < p.mlp_units) {
      for (int l = 1; l < p.n_layers; ++l) {
        const int out = p.dims[l + 1], in = p.dims[l];
        const int ncs = (out + 127) / 128, kbs = (in + 63) / 64;
        if (uu < ncs * kbs) { src = p.w[l]; rows = out; cols = in; nc = uu / kbs; kb = uu % kbs; break; }
        uu -= ncs * kbs;
      }
    } else {
      uu = u - p.mlp_units;
      const int K = p.dims[p.n_layers];
      const int kbs = (K + 63) / 64;
      src = p.codebook; rows = p.d; cols = K; nc = uu / kbs; kb = uu % kbs; transposed = true;  // B[n=j][k=code] = S[code][j]
    }
    const int n = nc * 128 + r;
    uint16_t v[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      const int k = kb * 64 + ch * 8 + e;
      uint16_t x = 0;
      if (n < rows && k < cols) x = transposed ? src[(size_t)k * rows + n] : src[(size_t)n * cols + k];
      v[e] = x;
    }
    uint4 q;
    q.x = v[0] | ((uint32_t)v[1] << 16); q.y = v[2] | ((uint32_t)v[3] << 16);
    q.z = v[4] | ((uint32_t)v[5] << 16); q.w = v[6] | ((uint32_t)v[7] << 16);
    *reinterpret_cast<uint4*>(p.units + (size_t)u * kUnitBytes + ((r >> 3) * 1024 + (r & 7) * 128 + ((ch ^ (r & 7)) << 4))) = q;
  }
  // constants
  const int h0 = p.dims[1], in = p.dims[0];
  for (int i = tid; i < h0 * in; i += nthreads) p.consts[i] = bf16_to_f32(p.w[0][i]);
  int off = h0 * in;
  for (int l = 0; l < p.n_layers; ++l) {
    const int out = p.dims[l + 1];
    for (int i = tid; i < out; i += nthreads) p.consts[off + i] = p.b[l] ? p.b[l][i] : 0.f;
    off += out;
  }
}

// ---------------------------------------------------------------------------------------------------------
// ---------------------------------------------------------------------------------------------------------
// Shared-memory plan (byte offsets from the 1024-aligned base; computed on the host, see plan_smem):
//   a_h     kbs_h units      A operand of the UMMA MLP layers (hidden activations, bf16, SW128 K-major)
//   a_p     2 x kbs_p units  A operand of the decode: probabilities of tile i in buffer i & 1
//   stage   8 x nbuf x 4 KB  per-epilogue-warp staging slabs [32 rows][64 bf16] (SW128) for the TMA tensor stores
//   ring    stages units     streamed B units
//   consts, barriers
struct SmemPlan {
  int a_h, a_p, stage, ring, consts, bars, total;
  int stages, nbuf, kbs_p;
  int a_in_tmem;  // decode A operand (probabilities) in TMEM columns [128,256) instead of shared memory
};

constexpr int kMaxStages = 8;
constexpr int kEpiWarps = 8;
constexpr int kSlabBytes = 4096;  // 32 rows x 128 B
constexpr int kBarBytes = 3072;   // mbarriers (first 512 B) + the softmax pair-exchange arrays [2][2][128] fp32

struct Barriers {
  uint64_t ring_full[kMaxStages], ring_empty[kMaxStages];
  uint64_t a_ready, acc_ready;
  uint64_t p_ready[2], p_empty[2];
  uint64_t dec_full[2], dec_empty[2];
  uint32_t tmem_base;
};

#ifdef LEGS_DECODE_TIMING
__device__ unsigned long long g_decode_wait[32];
#define LEGS_TWAIT(slot, ...)                           \
  do {                                                  \
    const long long t0__ = clock64();                   \
    __VA_ARGS__;                                        \
    tw__[(slot) & 3] += (unsigned long long)(clock64() - t0__); \
  } while (0)
#else
#define LEGS_TWAIT(slot, ...) __VA_ARGS__
#endif

struct DecodeArgs {
  DecodeParams p;
  SmemPlan s;
};

// Order in which B units are consumed (producer and MMA issuer walk it identically). Tile i of this CTA:
//   [i == 0: every UMMA layer of tile 0]  then  decode chunks 0..ncs-1 of tile i, with UMMA layer l of tile i+1
//   slotted in after chunk after(l) (so the MLP + softmax of the next tile overlap this tile's decode), and any
//   layer not yet issued after the last chunk.
__device__ __forceinline__ int layer_after_chunk(int l) { return 2 * l - 1; }  // layer 1 after chunk 1, layer 2 after 3

template <class FL, class FC, class FE>
__device__ __forceinline__ void walk_schedule(long long n_tiles, int n_umma, int ncs, FL&& on_layer, FC&& on_chunk,
                                              FE&& on_tile_end) {
  for (int l = 1; l <= n_umma; ++l) on_layer(l);
  for (long long i = 0; i < n_tiles; ++i) {
    const bool has_next = i + 1 < n_tiles;
    int next = 1;
    for (int nc = 0; nc < ncs; ++nc) {
      on_chunk(i, nc);
      while (has_next && next <= n_umma && nc == layer_after_chunk(next)) on_layer(next++);
    }
    on_tile_end(i);
    while (has_next && next <= n_umma) on_layer(next++);
  }
}

__global__ void __launch_bounds__(kThreads, 1) decode_kernel(const __grid_constant__ DecodeArgs args,
                                                             const __grid_constant__ CUtensorMap tmap_decoded,
                                                             const __grid_constant__ CUtensorMap tmap_probs) {
  extern __shared__ uint8_t smem_raw[];
#ifdef LEGS_DECODE_TIMING
  const long long t_start__ = clock64();
  unsigned long long tw__[4] = {0, 0, 0, 0};   // per-thread wait cycles, slot & 3
#endif
  const DecodeParams& p = args.p;
  const SmemPlan& sp = args.s;
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);  // 1024-aligned, still a shared pointer
  Barriers* bar = reinterpret_cast<Barriers*>(smem + sp.bars);
  float* s_consts = reinterpret_cast<float*>(smem + sp.consts);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int in_dim = p.dims[0], h0 = p.dims[1], K = p.dims[p.n_layers];
  const int n_umma = p.n_layers - 1;
  const bool dec = p.dec_units != 0;
  const int ncs = dec ? (p.d + 127) / 128 : 0;
  const int kbs_p = sp.kbs_p;
  const int stages = sp.stages;
  const long long my_tiles = (p.num_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x;

  if (threadIdx.x == 0) {
    for (int s = 0; s < stages; ++s) { mbar_init(&bar->ring_full[s], 1); mbar_init(&bar->ring_empty[s], 1); }
    mbar_init(&bar->a_ready, kFrontWarps * 32);
    mbar_init(&bar->acc_ready, 1);
    for (int b = 0; b < 2; ++b) {
      mbar_init(&bar->p_ready[b], kFrontWarps * 32);
      mbar_init(&bar->p_empty[b], 1);
      mbar_init(&bar->dec_full[b], 1);
      mbar_init(&bar->dec_empty[b], kEpiWarps);
    }
    fence_barrier_init();
    if (dec) prefetch_tmap(&tmap_decoded);
    if (p.probs) prefetch_tmap(&tmap_probs);
  }
  if (warp == 1) { tmem_alloc(&bar->tmem_base, kTmemCols); tmem_relinquish(); }
  {
    int nconst = h0 * in_dim;
    for (int l = 0; l < p.n_layers; ++l) nconst += p.dims[l + 1];
    for (int i = threadIdx.x; i < nconst; i += kThreads) s_consts[i] = p.consts[i];
  }
  fence_before_sync();
  __syncthreads();
  fence_after_sync();
  const uint32_t tmem = bar->tmem_base;

  // unit index (in p.units) of UMMA layer l, n-chunk nc, k-block kb
  auto layer_unit0 = [&](int l) {
    int off = 0;
    for (int j = 1; j < l; ++j) off += ((p.dims[j + 1] + 127) / 128) * ((p.dims[j] + 63) / 64);
    return off;
  };

  if (warp == 0) {
    // ===================== producer: stream B units through the ring in schedule order =====================
    if (lane == 0) {
      int s = 0; uint32_t ph = 0;
      auto push = [&](int u) {
        LEGS_TWAIT(0, mbar_wait(&bar->ring_empty[s], ph ^ 1));
        mbar_arrive_expect_tx(&bar->ring_full[s], kUnitBytes);
        bulk_g2s(smem + sp.ring + s * kUnitBytes, p.units + (size_t)u * kUnitBytes, kUnitBytes, &bar->ring_full[s]);
        if (++s == stages) { s = 0; ph ^= 1; }
      };
      walk_schedule(
          my_tiles, n_umma, ncs,
          [&](int l) {
            const int n = ((p.dims[l + 1] + 127) / 128) * ((p.dims[l] + 63) / 64), u0 = layer_unit0(l);
            for (int u = 0; u < n; ++u) push(u0 + u);
          },
          [&](long long, int nc) {
            for (int kb = 0; kb < kbs_p; ++kb) push(p.mlp_units + nc * kbs_p + kb);
          },
          [&](long long) {});
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    // The whole warp walks the schedule (uniform control flow, so descriptors and addresses live in uniform
    // registers); one elected lane issues the tcgen05.mma / tcgen05.commit instructions.
    int s = 0; uint32_t ph = 0;
    uint32_t a_par = 0, cc = 0;
    const uint32_t a_h_lo = desc_lo_sw128(smem_u32(smem + sp.a_h)), a_p_lo = desc_lo_sw128(smem_u32(smem + sp.a_p));
    const uint32_t ring_lo = desc_lo_sw128(smem_u32(smem + sp.ring));
    constexpr uint32_t kUnitLo = kUnitBytes >> 4;  // descriptor start-address units are 16 bytes
    // one B unit from the ring against k-block kb of the A operand, accumulating into d_tmem
    auto unit_mma = [&](uint32_t a_lo, uint32_t a_tmem, bool a_tm, int kb, int ktot, uint32_t d_tmem, uint32_t idesc) {
      LEGS_TWAIT(1, mbar_wait(&bar->ring_full[s], ph));
      fence_after_sync();
      const int ksteps = min(4, (ktot - kb * 64) >> 4);
      LEGS_TWAIT(2, if (elect_one_sync()) {
        const uint32_t al = a_lo + kb * kUnitLo, bl = ring_lo + s * kUnitLo;
        if (a_tm) {
          const uint32_t at = a_tmem + kb * 32;   // 32 columns per 64-wide k-block, 8 per K = 16 step
#pragma unroll
          for (int k = 0; k < 4; ++k)
            if (k < ksteps) umma_bf16_ts(d_tmem, at + 8 * k, bl + 2 * k, idesc, (kb | k) ? 1u : 0u);
        } else {
#pragma unroll
          for (int k = 0; k < 4; ++k)
            if (k < ksteps) umma_bf16_lo(d_tmem, al + 2 * k, bl + 2 * k, idesc, (kb | k) ? 1u : 0u);   // 32 bytes per K = 16 step
        }
        umma_commit(&bar->ring_empty[s]);
      }
      __syncwarp());
      if (++s == stages) { s = 0; ph ^= 1; }
    };
    walk_schedule(
        my_tiles, n_umma, ncs,
        [&](int l) {
          LEGS_TWAIT(3, mbar_wait(&bar->a_ready, a_par)); a_par ^= 1;   // A_h holds the input of layer l (and the
          fence_after_sync();                                            // accumulator columns have been drained)
          const int in = p.dims[l], out = p.dims[l + 1];
          const int lncs = (out + 127) / 128, lkbs = (in + 63) / 64;
          for (int nc = 0; nc < lncs; ++nc) {
            const uint32_t idesc = make_idesc_bf16(kRows, (uint32_t)min(128, out - nc * 128));
            for (int kb = 0; kb < lkbs; ++kb) unit_mma(a_h_lo, 0u, false, kb, in, tmem + nc * 128, idesc);
          }
          if (elect_one_sync()) umma_commit(&bar->acc_ready);
          __syncwarp();
        },
        [&](long long i, int nc) {
          const int pb = (int)(i & 1);
          if (nc == 0) { LEGS_TWAIT(3, mbar_wait(&bar->p_ready[pb], (uint32_t)((i >> 1) & 1))); fence_after_sync(); }
          const int b = cc & 1;
          LEGS_TWAIT(4, mbar_wait(&bar->dec_empty[b], ((cc >> 1) & 1) ^ 1)); ++cc;
          fence_after_sync();
          const uint32_t idesc = make_idesc_bf16(kRows, (uint32_t)min(128, p.d - nc * 128));
          for (int kb = 0; kb < kbs_p; ++kb)
            unit_mma(a_p_lo + pb * kbs_p * kUnitLo, tmem + kColAp + pb * 64, sp.a_in_tmem != 0, kb, K,
                     tmem + kColDecode + b * 128, idesc);
          if (elect_one_sync()) umma_commit(&bar->dec_full[b]);
          __syncwarp();
        },
        [&](long long i) {
          if (dec && elect_one_sync()) umma_commit(&bar->p_empty[i & 1]);
          __syncwarp();
        });
  } else if (warp < 2 + kFrontWarps) {
    // ===================== front group: 256 threads = 128 rows x 2 column halves ==================================
    // (layer 0 on the FP32 pipes, hidden epilogues, softmax -> A_p and probs). Warps w and w + 4 share a TMEM lane
    // quadrant and split the columns of every step; the softmax max and sum cross the pair through shared memory.
    const int row = 32 * (warp & 3) + lane;                    // TMEM lane this thread can read
    const int hf = (warp - 2) >> 2;                            // column half of this thread
    const uint32_t lane_addr = tmem + ((uint32_t)(32 * (warp & 3)) << 16);
    uint8_t* a_h = smem + sp.a_h;
    const float* W0 = s_consts;
    const float* bias0 = s_consts + h0 * in_dim;
    float* red_max = reinterpret_cast<float*>(smem + sp.bars + 512);   // [2][128]
    float* red_sum = red_max + 2 * kRows;                              // [2][128]
    uint32_t acc_par = 0;
    // feature row of the next tile, fetched one tile ahead
    uint4 fq0 = make_uint4(0, 0, 0, 0), fq1 = make_uint4(0, 0, 0, 0);
    auto fetch_feat = [&](long long t) {
      const long long r = t * kRows + row;
      fq0 = make_uint4(0, 0, 0, 0); fq1 = make_uint4(0, 0, 0, 0);
      if (r < p.P) {
        fq0 = *reinterpret_cast<const uint4*>(p.feat + r * in_dim);
        if (in_dim == 16) fq1 = *reinterpret_cast<const uint4*>(p.feat + r * in_dim + 8);
      }
    };
    fetch_feat(blockIdx.x);
    const bool store_leader = warp == 2 && lane == 0;   // issues the TMA stores of the probabilities
    const bool need_ap_smem = p.probs != nullptr || !sp.a_in_tmem;   // A_p tile in shared memory: TMA-store source / A operand
    for (long long i = 0; i < my_tiles; ++i) {
      const long long tile = blockIdx.x + i * gridDim.x;
      // ---- layer 0: h = relu(W0 x + b0) -> A_h (bf16, swizzled); this thread's half of the 16-byte chunks
      float x[16];
      {
        const uint32_t w[8] = {fq0.x, fq0.y, fq0.z, fq0.w, fq1.x, fq1.y, fq1.z, fq1.w};
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          x[2 * k] = __uint_as_float(w[k] << 16);
          x[2 * k + 1] = __uint_as_float(w[k] & 0xffff0000u);
        }
      }
      for (int c = hf; c < h0 / 8; c += 2) {
        float h[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
          const float4* wr = reinterpret_cast<const float4*>(W0 + (c * 8 + e) * in_dim);
          float acc = bias0[c * 8 + e];
          const float4 w0 = wr[0], w1 = wr[1];
          acc = fmaf(w0.x, x[0], acc); acc = fmaf(w0.y, x[1], acc); acc = fmaf(w0.z, x[2], acc); acc = fmaf(w0.w, x[3], acc);
          acc = fmaf(w1.x, x[4], acc); acc = fmaf(w1.y, x[5], acc); acc = fmaf(w1.z, x[6], acc); acc = fmaf(w1.w, x[7], acc);
          if (in_dim == 16) {
            const float4 w2 = wr[2], w3 = wr[3];
            acc = fmaf(w2.x, x[8], acc); acc = fmaf(w2.y, x[9], acc); acc = fmaf(w2.z, x[10], acc); acc = fmaf(w2.w, x[11], acc);
            acc = fmaf(w3.x, x[12], acc); acc = fmaf(w3.y, x[13], acc); acc = fmaf(w3.z, x[14], acc); acc = fmaf(w3.w, x[15], acc);
          }
          h[e] = fmaxf(acc, 0.f);
        }
        const uint4 q = make_uint4(pack_bf16(h[0], h[1]), pack_bf16(h[2], h[3]), pack_bf16(h[4], h[5]), pack_bf16(h[6], h[7]));
        *reinterpret_cast<uint4*>(a_h + (c >> 3) * kUnitBytes + sw128_offset(row, c & 7)) = q;
      }
      fence_proxy_async_smem();
      mbar_arrive(&bar->a_ready);
      if (i + 1 < my_tiles) fetch_feat(tile + gridDim.x);
      // ---- UMMA layers: hidden ones -> bias, ReLU -> A_h ; last one -> softmax -> A_p (+ probs)
      int boff = h0 * in_dim + h0;
      for (int l = 1; l <= n_umma; ++l) {
        const int out = p.dims[l + 1];
        const float* bias = s_consts + boff;
        boff += out;
        LEGS_TWAIT(0, mbar_wait(&bar->acc_ready, acc_par)); acc_par ^= 1;
        fence_after_sync();
        if (l < n_umma) {
          for (int g = hf; g < out / 32; g += 2) {
            uint32_t r[32];
            tmem_ld32(lane_addr + g * 32, r);
            tmem_ld_wait();
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              float h[8];
#pragma unroll
              for (int e = 0; e < 8; ++e) h[e] = fmaxf(__uint_as_float(r[c * 8 + e]) + bias[g * 32 + c * 8 + e], 0.f);
              const uint4 q = make_uint4(pack_bf16(h[0], h[1]), pack_bf16(h[2], h[3]), pack_bf16(h[4], h[5]), pack_bf16(h[6], h[7]));
              const int chunk = g * 4 + c;  // 16-byte chunk index along k
              *reinterpret_cast<uint4*>(a_h + (chunk >> 3) * kUnitBytes + sw128_offset(row, chunk & 7)) = q;
            }
          }
          fence_before_sync();
          fence_proxy_async_smem();
          mbar_arrive(&bar->a_ready);
        } else {
          // softmax over K <= 128 logits; this thread holds the 32-column groups g = hf, hf + 2 (at most two)
          const int ng = K / 32;
          const float kLog2e = 1.4426950408889634f;
          // three passes of 32 columns (max; exp parked in TMEM over the logits; scale) keep the live registers low
          float mx = -3.0e38f;
          for (int g = hf; g < ng; g += 2) {
            uint32_t r[32];
            tmem_ld32(lane_addr + g * 32, r);
            tmem_ld_wait();
            float m4[4] = {-3.0e38f, -3.0e38f, -3.0e38f, -3.0e38f};
#pragma unroll
            for (int e = 0; e < 32; ++e) m4[e & 3] = fmaxf(m4[e & 3], __uint_as_float(r[e]) + bias[g * 32 + e]);
            mx = fmaxf(mx, fmaxf(fmaxf(m4[0], m4[1]), fmaxf(m4[2], m4[3])));
          }
          red_max[hf * kRows + row] = mx;
          asm volatile("bar.sync 1, %0;" ::"n"(kFrontWarps * 32) : "memory");
          mx = fmaxf(mx, red_max[(hf ^ 1) * kRows + row]);
          const float mxs = mx * kLog2e;
          float s4[4] = {0.f, 0.f, 0.f, 0.f};
          for (int g = hf; g < ng; g += 2) {
            uint32_t r[32];
            tmem_ld32(lane_addr + g * 32, r);
            tmem_ld_wait();
#pragma unroll
            for (int e = 0; e < 32; ++e) {
              float ex;
              asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(ex) : "f"(fmaf(__uint_as_float(r[e]) + bias[g * 32 + e], kLog2e, -mxs)));
              r[e] = __float_as_uint(ex);
              s4[e & 3] += ex;
            }
            tmem_st32(lane_addr + g * 32, r);
          }
          tmem_st_wait();
          const float part = (s4[0] + s4[1]) + (s4[2] + s4[3]);
          red_sum[hf * kRows + row] = part;
          // A_p[i & 1] is rewritten below: its probability stores of tile i-2 must have finished reading it
          if (store_leader && p.probs) bulk_wait_read<1>();
          asm volatile("bar.sync 1, %0;" ::"n"(kFrontWarps * 32) : "memory");
          const float inv = 1.0f / (part + red_sum[(hf ^ 1) * kRows + row]);
          uint8_t* a_p = smem + sp.a_p + (int)(i & 1) * kbs_p * kUnitBytes;
          if (dec && i >= 2) LEGS_TWAIT(1, mbar_wait(&bar->p_empty[i & 1], (uint32_t)(((i >> 1) - 1) & 1)));  // decode of tile i-2 done
          for (int g = hf; g < ng; g += 2) {
            uint32_t r[32];
            tmem_ld32(lane_addr + g * 32, r);
            tmem_ld_wait();
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              const uint4 q = make_uint4(
                  pack_bf16(__uint_as_float(r[c * 8]) * inv, __uint_as_float(r[c * 8 + 1]) * inv),
                  pack_bf16(__uint_as_float(r[c * 8 + 2]) * inv, __uint_as_float(r[c * 8 + 3]) * inv),
                  pack_bf16(__uint_as_float(r[c * 8 + 4]) * inv, __uint_as_float(r[c * 8 + 5]) * inv),
                  pack_bf16(__uint_as_float(r[c * 8 + 6]) * inv, __uint_as_float(r[c * 8 + 7]) * inv));
              const int chunk = g * 4 + c;
              if (need_ap_smem) *reinterpret_cast<uint4*>(a_p + (chunk >> 3) * kUnitBytes + sw128_offset(row, chunk & 7)) = q;
              r[c * 4] = q.x; r[c * 4 + 1] = q.y; r[c * 4 + 2] = q.z; r[c * 4 + 3] = q.w;
            }
            if (sp.a_in_tmem) {   // packed pairs: K elements 32g .. 32g+31 -> columns 16g .. 16g+15 of this buffer
              const uint32_t (&r16)[16] = reinterpret_cast<const uint32_t (&)[16]>(r);
              tmem_st16(lane_addr + kColAp + (uint32_t)(i & 1) * 64 + g * 16, r16);
            }
          }
          if (sp.a_in_tmem) tmem_st_wait();
          fence_before_sync();
          fence_proxy_async_smem();
          mbar_arrive(&bar->p_ready[i & 1]);
          if (store_leader && p.probs) {
            // the A_p tile is the probability tile in the TMA 128-byte-swizzled box layout: one tensor store per k-block
            mbar_wait(&bar->p_ready[i & 1], (uint32_t)((i >> 1) & 1));
            for (int kb = 0; kb < kbs_p; ++kb) tma_store_2d(&tmap_probs, a_p + kb * kUnitBytes, kb * 64, (int32_t)(tile * kRows));
            bulk_commit();
          }
        }
      }
    }
    if (store_leader && p.probs) bulk_wait<0>();
  } else {
    // ===================== epilogue group: 8 warps, TMEM -> bf16 -> swizzled slab -> TMA tensor store ==============
    const int ew = warp - 2 - kFrontWarps;  // 0..7
    const int q = warp & 3;               // TMEM lane quadrant this warp can read
    const int half = ew >> 2;             // which 64 of the chunk's 128 columns
    const uint32_t lane_addr = tmem + ((uint32_t)(32 * q) << 16) + kColDecode + half * 64;
    uint8_t* slab0 = smem + sp.stage + ew * sp.nbuf * kSlabBytes;
    const uint32_t swz = (uint32_t)(lane >> 3) * 1024u + (uint32_t)(lane & 7) * 128u;
    uint32_t cc = 0, stores = 0;
    if (dec) {
      for (long long i = 0; i < my_tiles; ++i) {
        const long long tile = blockIdx.x + i * gridDim.x;
        for (int nc = 0; nc < ncs; ++nc, ++cc) {
          const int b = cc & 1;
          LEGS_TWAIT(0, mbar_wait(&bar->dec_full[b], (cc >> 1) & 1));
          fence_after_sync();
          const bool have = nc * 128 + half * 64 < p.d;
          uint8_t* slab = slab0 + (sp.nbuf == 2 ? (int)(stores & 1) * kSlabBytes : 0);
          uint32_t r0[32], r1[32];
          LEGS_TWAIT(2, if (have) {
            tmem_ld32(lane_addr + b * 128, r0);
            tmem_ld32(lane_addr + b * 128 + 32, r1);
            tmem_ld_wait();
          }
          // the accumulator buffer is free as soon as it is in registers: release it before converting and storing
          fence_before_sync();
          __syncwarp();
          if (lane == 0) mbar_arrive(&bar->dec_empty[b]));
          if (have) {
            ++stores;
            if (lane == 0) {  // the slab's previous store must have finished reading shared memory
              LEGS_TWAIT(1, if (sp.nbuf == 2) bulk_wait_read<1>(); else bulk_wait_read<0>());
            }
            __syncwarp();
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              const uint4 v = make_uint4(pack_bf16(__uint_as_float(r0[c * 8]), __uint_as_float(r0[c * 8 + 1])),
                                         pack_bf16(__uint_as_float(r0[c * 8 + 2]), __uint_as_float(r0[c * 8 + 3])),
                                         pack_bf16(__uint_as_float(r0[c * 8 + 4]), __uint_as_float(r0[c * 8 + 5])),
                                         pack_bf16(__uint_as_float(r0[c * 8 + 6]), __uint_as_float(r0[c * 8 + 7])));
              *reinterpret_cast<uint4*>(slab + swz + (((uint32_t)c ^ (uint32_t)(lane & 7)) << 4)) = v;
            }
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              const uint4 v = make_uint4(pack_bf16(__uint_as_float(r1[c * 8]), __uint_as_float(r1[c * 8 + 1])),
                                         pack_bf16(__uint_as_float(r1[c * 8 + 2]), __uint_as_float(r1[c * 8 + 3])),
                                         pack_bf16(__uint_as_float(r1[c * 8 + 4]), __uint_as_float(r1[c * 8 + 5])),
                                         pack_bf16(__uint_as_float(r1[c * 8 + 6]), __uint_as_float(r1[c * 8 + 7])));
              *reinterpret_cast<uint4*>(slab + swz + (((uint32_t)(c + 4) ^ (uint32_t)(lane & 7)) << 4)) = v;
            }
          }
          if (!have) continue;
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            tma_store_2d(&tmap_decoded, slab, nc * 128 + half * 64, (int32_t)(tile * kRows + 32 * q));
            bulk_commit();
          }
        }
      }
      if (lane == 0) bulk_wait<0>();
    }
  }
  fence_before_sync();
  __syncthreads();
  if (warp == 1) { fence_after_sync(); tmem_dealloc(tmem, kTmemCols); }
#ifdef LEGS_DECODE_TIMING
  if (blockIdx.x == 0) {   // rows: 0 producer, 1 issuer, 2 front warp 2, 3 epilogue warp 6, 4 epilogue warp 10; 4 slots each
    const int rowi = threadIdx.x == 0 ? 0 : threadIdx.x == 32 ? 1 : threadIdx.x == 64 ? 2 : threadIdx.x == 320 ? 3 : threadIdx.x == 448 ? 4 : -1;
    if (rowi >= 0) for (int k = 0; k < 4; ++k) g_decode_wait[rowi * 4 + k] = tw__[k];
    if (threadIdx.x == 0) { g_decode_wait[31] = (unsigned long long)(clock64() - t_start__); g_decode_wait[30] = (unsigned long long)my_tiles; }
  }
#endif
}

// Host: carve the shared memory of decode_kernel. Returns false if the decoder does not fit.
bool plan_smem(const DecodeParams& p, SmemPlan* out) {
  const int n_umma = p.n_layers - 1;
  int kbs_h = 1;
  for (int l = 1; l <= n_umma; ++l) kbs_h = std::max(kbs_h, (p.dims[l] + 63) / 64);
  const int kbs_p = (p.dims[p.n_layers] + 63) / 64;
  int max_out = 0;
  for (int l = 1; l <= n_umma; ++l) max_out = std::max(max_out, p.dims[l + 1]);
  const int a_in_tmem = max_out <= kColAp ? 1 : 0;
  int nconst = p.dims[0] * p.dims[1];
  for (int l = 0; l < p.n_layers; ++l) nconst += p.dims[l + 1];
  const int consts_bytes = (int)legs_align_up((size_t)nconst * 4, 1024);
  const int fixed = (kbs_h + 2 * kbs_p) * kUnitBytes + consts_bytes + kBarBytes;
  const int budget = 227 * 1024 - 1024;  // 1 KB of slack for the base alignment
  int nbuf = 2;
  int stages = (budget - fixed - kEpiWarps * nbuf * kSlabBytes) / kUnitBytes;
  if (stages < 3) { nbuf = 1; stages = (budget - fixed - kEpiWarps * nbuf * kSlabBytes) / kUnitBytes; }
  if (stages < 2) return false;
  stages = std::min(stages, kMaxStages);
  SmemPlan s;
  s.a_h = 0;
  s.a_p = kbs_h * kUnitBytes;
  s.stage = s.a_p + 2 * kbs_p * kUnitBytes;
  s.ring = s.stage + kEpiWarps * nbuf * kSlabBytes;
  s.consts = s.ring + stages * kUnitBytes;
  s.bars = s.consts + consts_bytes;
  s.total = s.bars + kBarBytes;
  s.stages = stages; s.nbuf = nbuf; s.kbs_p = kbs_p;
  s.a_in_tmem = a_in_tmem;
  *out = s;
  return true;
}

int count_units(const legs_decoder* dec, int d, int* mlp_units, int* dec_units) {
  const int dims[4] = {dec->in_dim, dec->hidden[0], dec->n_layers == 3 ? dec->hidden[1] : dec->n_codes, dec->n_codes};
  int mu = 0;
  for (int l = 1; l < dec->n_layers; ++l) mu += ((dims[l + 1] + 127) / 128) * ((dims[l] + 63) / 64);
  *mlp_units = mu;
  *dec_units = ((d + 127) / 128) * ((dec->n_codes + 63) / 64);
  return 0;
}

int check_decoder(const legs_decoder* dec, int d) {
  if (!dec) return LEGS_ERR_NULL;
  if (dec->n_layers != 2 && dec->n_layers != 3) return LEGS_ERR_DIM;
  if (dec->in_dim != 8 && dec->in_dim != 16) return LEGS_ERR_DIM;
  for (int l = 0; l < dec->n_layers - 1; ++l)
    if (dec->hidden[l] < 32 || dec->hidden[l] > kMaxHidden || (dec->hidden[l] % 32)) return LEGS_ERR_DIM;
  if (dec->n_codes != 32 && dec->n_codes != 64 && dec->n_codes != 128) return LEGS_ERR_DIM;
  if (d < 64 || d > 1024 || (d % 64)) return LEGS_ERR_DIM;
  for (int l = 0; l < dec->n_layers; ++l) {
    if (!dec->w[l]) return LEGS_ERR_NULL;
    if (!legs_aligned16(dec->w[l]) || (dec->b[l] && !legs_aligned16(dec->b[l]))) return LEGS_ERR_ALIGN;
  }
  return LEGS_OK;
}

size_t consts_floats(const legs_decoder* dec) {
  size_t n = (size_t)dec->hidden[0] * dec->in_dim + dec->hidden[0] + dec->n_codes;
  if (dec->n_layers == 3) n += dec->hidden[1];
  return n;
}

}  // namespace

extern "C" {

#ifdef LEGS_DECODE_TIMING
// measurement builds only (not declared in legs.h): cycles block 0 spent in each pipeline wait, then resets them
int legs_debug_decode_waits(unsigned long long* out32) {
  if (cudaMemcpyFromSymbol(out32, g_decode_wait, sizeof(g_decode_wait)) != cudaSuccess) return LEGS_ERR_CUDA;
  unsigned long long z[32] = {0};
  return cudaMemcpyToSymbol(g_decode_wait, z, sizeof(z)) == cudaSuccess ? LEGS_OK : LEGS_ERR_CUDA;
}
#endif

size_t legs_decode_workspace_bytes(const legs_decoder* dec, int32_t d) {
  if (check_decoder(dec, d) != LEGS_OK) return 0;
  int mu, du;
  count_units(dec, d, &mu, &du);
  return (size_t)(mu + du) * kUnitBytes + legs_align_up(consts_floats(dec) * 4, 256);
}

// Packs the decoder weights and the codebook into the workspace (B units in consumption order + fp32 constants).
int legs_decode_prepare(legs_ctx* ctx, const legs_decoder* dec, const uint16_t* codebook, int32_t d, void* workspace,
                        size_t workspace_bytes, void* stream) {
  if (!ctx) return LEGS_ERR_NULL;
  int rc;
  if ((rc = check_decoder(dec, d)) != LEGS_OK) return rc;
  if (!codebook || !workspace) return LEGS_ERR_NULL;
  if (!legs_aligned16(codebook) || !legs_aligned16(workspace)) return LEGS_ERR_ALIGN;
  if (workspace_bytes < legs_decode_workspace_bytes(dec, d)) return LEGS_ERR_WORKSPACE;
  int mu, du;
  count_units(dec, d, &mu, &du);
  PackParams pp;
  pp.n_layers = dec->n_layers;
  pp.dims[0] = dec->in_dim; pp.dims[1] = dec->hidden[0];
  pp.dims[2] = dec->n_layers == 3 ? dec->hidden[1] : dec->n_codes;
  pp.dims[3] = dec->n_codes;
  pp.d = d;
  for (int l = 0; l < 3; ++l) { pp.w[l] = l < dec->n_layers ? dec->w[l] : nullptr; pp.b[l] = l < dec->n_layers ? dec->b[l] : nullptr; }
  pp.codebook = codebook;
  pp.units = (uint8_t*)workspace;
  pp.consts = (float*)((uint8_t*)workspace + (size_t)(mu + du) * kUnitBytes);
  pp.mlp_units = mu; pp.dec_units = du;
  pack_kernel<<<64, 256, 0, (cudaStream_t)stream>>>(pp);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

int legs_decode_semantics_packed(legs_ctx* ctx, const uint16_t* feat, int64_t P, const legs_decoder* dec, int32_t d,
                                 uint16_t* probs, uint16_t* decoded, const void* workspace, size_t workspace_bytes,
                                 void* stream) {
  if (!ctx) return LEGS_ERR_NULL;
  int rc;
  if ((rc = check_decoder(dec, d)) != LEGS_OK) return rc;
  if (!feat || !workspace) return LEGS_ERR_NULL;
  if (!legs_aligned16(feat) || !legs_aligned16(workspace) || (probs && !legs_aligned16(probs)) ||
      (decoded && !legs_aligned16(decoded)))
    return LEGS_ERR_ALIGN;
  if (P < 0) return LEGS_ERR_DIM;
  if (workspace_bytes < legs_decode_workspace_bytes(dec, d)) return LEGS_ERR_WORKSPACE;
  if (P == 0 || (!probs && !decoded)) return LEGS_OK;
  cudaStream_t st = (cudaStream_t)stream;
  int mu, du_full;
  count_units(dec, d, &mu, &du_full);
  DecodeParams dp;
  dp.P = P; dp.n_layers = dec->n_layers;
  dp.dims[0] = dec->in_dim; dp.dims[1] = dec->hidden[0];
  dp.dims[2] = dec->n_layers == 3 ? dec->hidden[1] : dec->n_codes;
  dp.dims[3] = dec->n_codes;
  dp.d = d; dp.mlp_units = mu; dp.dec_units = decoded ? du_full : 0;
  dp.feat = feat; dp.units = (const uint8_t*)workspace;
  dp.consts = (const float*)((const uint8_t*)workspace + (size_t)(mu + du_full) * kUnitBytes);
  dp.probs = probs; dp.decoded = decoded;
  dp.num_tiles = (P + kRows - 1) / kRows;
  DecodeArgs args;
  args.p = dp;
  if (!plan_smem(dp, &args.s)) return LEGS_ERR_DIM;
  // tensor maps: decoded [P, d] bf16 with a 64-column x 32-row box (one epilogue-warp slab), probs [P, K] bf16 with
  // a 64-column x 128-row box (one k-block of the A_p tile); both 128-byte swizzled
  CUtensorMap tmap_dec, tmap_pr;
  memset(&tmap_dec, 0, sizeof(tmap_dec));
  memset(&tmap_pr, 0, sizeof(tmap_pr));
  if (decoded && (rc = make_tmap_bf16_2d(ctx, decoded, (uint64_t)d, (uint64_t)P, 64, 32, &tmap_dec)) != LEGS_OK) return rc;
  if (probs && (rc = make_tmap_bf16_2d(ctx, probs, (uint64_t)dec->n_codes, (uint64_t)P, 64, kRows, &tmap_pr)) != LEGS_OK)
    return rc;
  const int smem_bytes = args.s.total + 1024;
  LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(decode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
  const int grid = (int)(dp.num_tiles < ctx->num_sms ? dp.num_tiles : ctx->num_sms);
  decode_kernel<<<grid, kThreads, smem_bytes, st>>>(args, tmap_dec, tmap_pr);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

int legs_decode_semantics(legs_ctx* ctx, const uint16_t* feat, int64_t P, const legs_decoder* dec,
                          const uint16_t* codebook, int32_t d, uint16_t* probs, uint16_t* decoded, void* workspace,
                          size_t workspace_bytes, void* stream) {
  if (!ctx) return LEGS_ERR_NULL;
  if (!feat) return LEGS_ERR_NULL;
  if (!legs_aligned16(feat) || (probs && !legs_aligned16(probs)) || (decoded && !legs_aligned16(decoded))) return LEGS_ERR_ALIGN;
  if (P < 0) return LEGS_ERR_DIM;
  int rc;
  if ((rc = legs_decode_prepare(ctx, dec, codebook, d, workspace, workspace_bytes, stream)) != LEGS_OK) return rc;
  return legs_decode_semantics_packed(ctx, feat, P, dec, d, probs, decoded, workspace, workspace_bytes, stream);
}

}  // extern "C"

// =========================================================================================================
// S11 relevancy from probabilities (Gram shortcut): with F = p^T S and S_c = S[:, 0:d_clip],
//   |F_clip|^2 = p^T (S_c S_c^T) p,   F_clip . q = p^T (S_c q)
// so the decoded map is never read. Per 128-pixel tile one UMMA computes Y = P [G | V] (G = S_c S_c^T in bf16,
// V = S_c q / |q|), the row threads finish with sum_k Y_k p_k and the division.
namespace {

constexpr int kRelThreads = 320;  // warp 0: TMA producer, warp 1: MMA issuer + TMEM, warps 2-9: two epilogue groups
constexpr int kRelQPad = 16;

struct RelParams {
  long long P, num_tiles;
  int K, Q;
  const uint16_t* probs;
  const uint8_t* units;  // [G kb0, G kb1, V kb0, V kb1] bf16 units (kb1 absent when K <= 64)
  float* rel;
};

// G[n][k] = <S_n[0:dc], S_k[0:dc]>, V[q][k] = <S_k[0:dc], query_q> / |query_q| -> bf16 B units
__global__ void __launch_bounds__(128) rel_pack_kernel(const uint16_t* __restrict__ codebook, int K, int d, int d_clip,
                                                       const uint16_t* __restrict__ queries, int Q, uint8_t* units) {
  __shared__ float s_a[1024];          // this block's row (a codebook row or a query), fp32
  __shared__ float s_nq[4];
  const int kbs = (K + 63) / 64;
  const int row = blockIdx.x;  // 0..K-1: G rows; K..K+kRelQPad-1: V rows
  const bool is_v = row >= K;
  const int n = is_v ? row - K : row;
  const bool live = !is_v || n < Q;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint16_t* a = is_v ? queries + (size_t)n * d_clip : codebook + (size_t)n * d;
  float nq = 0.f;
  for (int t = threadIdx.x; t < d_clip; t += 128) {
    const float av = live ? bf16_to_f32(a[t]) : 0.f;
    s_a[t] = av;
    nq = fmaf(av, av, nq);
  }
  for (int o = 16; o > 0; o >>= 1) nq += __shfl_xor_sync(0xffffffffu, nq, o);
  if (lane == 0) s_nq[warp] = nq;
  __syncthreads();
  const float scale = is_v ? rsqrtf((s_nq[0] + s_nq[1]) + (s_nq[2] + s_nq[3])) : 1.0f;
  // one warp per codebook row k: lanes stride over the d_clip dimensions (coalesced), then a warp reduction
  for (int k = warp; k < kbs * 64; k += 4) {
    float acc = 0.f;
    if (k < K && live) {
      const uint16_t* b = codebook + (size_t)k * d;
      for (int t = lane; t < d_clip; t += 32) acc = fmaf(s_a[t], bf16_to_f32(b[t]), acc);
    }
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) {
      if (is_v) acc *= scale;
      const int kb = k / 64, ch = (k % 64) / 8, e = k % 8;
      const int u = (is_v ? kbs : 0) + kb;
      uint16_t* dst = reinterpret_cast<uint16_t*>(units + (size_t)u * kUnitBytes + sw128_offset((uint32_t)n, (uint32_t)ch)) + e;
      *dst = (uint16_t)(pack_bf16(k < K && live ? acc : 0.f, 0.f) & 0xffffu);
    }
  }
}

constexpr int kRelStages = 4;           // probability tiles in flight (TMA ring)
constexpr int kRelAccStride = 256;      // TMEM columns per accumulator buffer: [0,128) Y = P G, [128,144) P V

struct RelBarriers {
  uint64_t full[kRelStages], empty[kRelStages];
  uint64_t acc_full[2], acc_empty[2];
  uint32_t tmem_base;
};

// Persistent, one CTA per SM. warp 0: TMA producer (probability tiles land directly in the UMMA A layout), warp 1: MMA
// issuer + TMEM, warps 2-5 / 6-9: two epilogue groups that alternate tiles (one TMEM accumulator buffer each), so the
// loads, the MMAs of tile i+1 and the finishing arithmetic of tile i overlap. HBM-bound: 2 K bytes read per pixel.
__global__ void __launch_bounds__(kRelThreads, 1) relevancy_kernel(const __grid_constant__ RelParams p,
                                                                   const __grid_constant__ CUtensorMap tmap_probs) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const int K = p.K, kbs = (K + 63) / 64;
  uint8_t* b_u = smem;                                   // 2 * kbs resident B units: G then V
  uint8_t* ring = smem + 2 * kbs * kUnitBytes;           // kRelStages x kbs units
  RelBarriers* bar = reinterpret_cast<RelBarriers*>(ring + kRelStages * kbs * kUnitBytes);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long my_tiles = (p.num_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x;
  if (threadIdx.x == 0) {
    for (int s = 0; s < kRelStages; ++s) { mbar_init(&bar->full[s], 1); mbar_init(&bar->empty[s], 5); }
    for (int b = 0; b < 2; ++b) { mbar_init(&bar->acc_full[b], 1); mbar_init(&bar->acc_empty[b], 4); }
    fence_barrier_init();
    prefetch_tmap(&tmap_probs);
  }
  if (warp == 1) { tmem_alloc(&bar->tmem_base, 512); tmem_relinquish(); }
  for (int i = threadIdx.x; i < 2 * kbs * (kUnitBytes / 16); i += kRelThreads)
    reinterpret_cast<uint4*>(b_u)[i] = reinterpret_cast<const uint4*>(p.units)[i];
  fence_proxy_async_smem();
  fence_before_sync();
  __syncthreads();
  fence_after_sync();
  const uint32_t tmem = bar->tmem_base;

  if (warp == 0) {
    if (lane == 0) {
      int s = 0; uint32_t ph = 0;
      for (long long i = 0; i < my_tiles; ++i) {
        const long long tile = blockIdx.x + i * gridDim.x;
        mbar_wait(&bar->empty[s], ph ^ 1);
        mbar_arrive_expect_tx(&bar->full[s], (uint32_t)(kbs * kUnitBytes));
        for (int kb = 0; kb < kbs; ++kb)
          tma_load_2d(ring + (s * kbs + kb) * kUnitBytes, &tmap_probs, kb * 64, (int32_t)(tile * kRows), &bar->full[s]);
        if (++s == kRelStages) { s = 0; ph ^= 1; }
      }
    }
  } else if (warp == 1) {
    int s = 0; uint32_t ph = 0;
    const uint32_t b_lo = desc_lo_sw128(smem_u32(b_u)), ring_lo = desc_lo_sw128(smem_u32(ring));
    constexpr uint32_t kUnitLo = kUnitBytes >> 4;
    const uint32_t idesc_g = make_idesc_bf16(kRows, (uint32_t)K), idesc_v = make_idesc_bf16(kRows, kRelQPad);
    for (long long i = 0; i < my_tiles; ++i) {
      const int b = (int)(i & 1);
      mbar_wait(&bar->full[s], ph);
      mbar_wait(&bar->acc_empty[b], (uint32_t)(((i >> 1) & 1) ^ 1));
      fence_after_sync();
      if (elect_one_sync()) {
        const uint32_t d = tmem + b * kRelAccStride;
        for (int kb = 0; kb < kbs; ++kb) {
          const int ksteps = min(4, (K - kb * 64) >> 4);
          const uint32_t al = ring_lo + (s * kbs + kb) * kUnitLo;
          for (int k = 0; k < ksteps; ++k) {
            umma_bf16_lo(d, al + 2 * k, b_lo + kb * kUnitLo + 2 * k, idesc_g, (kb | k) ? 1u : 0u);
            umma_bf16_lo(d + 128, al + 2 * k, b_lo + (kbs + kb) * kUnitLo + 2 * k, idesc_v, (kb | k) ? 1u : 0u);
          }
        }
        umma_commit(&bar->empty[s]);       // one of the stage's five releases (the epilogue warps give the others)
        umma_commit(&bar->acc_full[b]);
      }
      __syncwarp();
      if (++s == kRelStages) { s = 0; ph ^= 1; }
    }
  } else {
    const int grp = (warp - 2) >> 2;                           // epilogue group = accumulator buffer
    const int row = 32 * (warp & 3) + lane;
    const uint32_t lane_addr = tmem + ((uint32_t)(32 * (warp & 3)) << 16) + grp * kRelAccStride;
    for (long long i = grp; i < my_tiles; i += 2) {
      const long long tile = blockIdx.x + i * gridDim.x;
      const long long prow = tile * kRows + row;
      const int s = (int)(i % kRelStages);
      const uint32_t ph = (uint32_t)((i / kRelStages) & 1);
      mbar_wait(&bar->full[s], ph);                            // the probability tile (read below with plain loads)
      mbar_wait(&bar->acc_full[grp], (uint32_t)((i >> 1) & 1));
      fence_after_sync();
      const uint8_t* a_p = ring + s * kbs * kUnitBytes;
      float n4[4] = {0.f, 0.f, 0.f, 0.f};
      for (int g = 0; g < K / 32; ++g) {
        uint32_t r[32];
        tmem_ld32(lane_addr + g * 32, r);
        uint4 pr[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const int chunk = g * 4 + c;
          pr[c] = *reinterpret_cast<const uint4*>(a_p + (chunk >> 3) * kUnitBytes + sw128_offset(row, chunk & 7));
        }
        tmem_ld_wait();
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const uint32_t w[4] = {pr[c].x, pr[c].y, pr[c].z, pr[c].w};
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            n4[e] = fmaf(__uint_as_float(r[c * 8 + 2 * e]), __uint_as_float(w[e] << 16), n4[e]);
            n4[e] = fmaf(__uint_as_float(r[c * 8 + 2 * e + 1]), __uint_as_float(w[e] & 0xffff0000u), n4[e]);
          }
        }
      }
      uint32_t dots[16];
      tmem_ld16(lane_addr + 128, dots);
      tmem_ld_wait();
      fence_before_sync();
      __syncwarp();
      if (lane == 0) { mbar_arrive(&bar->acc_empty[grp]); mbar_arrive(&bar->empty[s]); }
      if (prow < p.P) {
        const float norm2 = (n4[0] + n4[1]) + (n4[2] + n4[3]);
        const float inv = rsqrtf(fmaxf(norm2, 1e-30f));
        if (p.Q == 4) {
          *reinterpret_cast<float4*>(p.rel + prow * 4) = make_float4(__uint_as_float(dots[0]) * inv, __uint_as_float(dots[1]) * inv,
                                                                    __uint_as_float(dots[2]) * inv, __uint_as_float(dots[3]) * inv);
        } else {
#pragma unroll
          for (int q = 0; q < kRelQPad; ++q)
            if (q < p.Q) p.rel[prow * p.Q + q] = __uint_as_float(dots[q]) * inv;
        }
      }
    }
  }
  fence_before_sync();
  __syncthreads();
  if (warp == 1) { fence_after_sync(); tmem_dealloc(tmem, 512); }
}

}  // namespace

extern "C" {

size_t legs_relevancy_workspace_bytes(int32_t K, int32_t Q) {
  (void)Q;
  return (size_t)2 * ((K + 63) / 64) * kUnitBytes;
}

// Packs G = S_c S_c^T and V = S_c q / |q| (bf16 B units) into the workspace.
int legs_relevancy_prepare(legs_ctx* ctx, const uint16_t* codebook, int32_t K, int32_t d, int32_t d_clip,
                           const uint16_t* queries, int32_t Q, void* workspace, size_t workspace_bytes, void* stream) {
  if (!ctx || !codebook || !queries || !workspace) return LEGS_ERR_NULL;
  if (!legs_aligned16(codebook) || !legs_aligned16(queries) || !legs_aligned16(workspace)) return LEGS_ERR_ALIGN;
  // the pack kernel stages one row of d_clip floats in 4 KB of shared memory
  if ((K != 32 && K != 64 && K != 128) || Q < 1 || Q > kRelQPad || d_clip < 1 || d_clip > d || d_clip > 1024) return LEGS_ERR_DIM;
  if (workspace_bytes < legs_relevancy_workspace_bytes(K, Q)) return LEGS_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  LEGS_CUDA_CHECK(ctx, cudaMemsetAsync(workspace, 0, legs_relevancy_workspace_bytes(K, Q), st));
  rel_pack_kernel<<<K + kRelQPad, 128, 0, st>>>(codebook, K, d, d_clip, queries, Q, (uint8_t*)workspace);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

int legs_relevancy_packed(legs_ctx* ctx, const uint16_t* probs, int64_t P, int32_t K, int32_t Q, float* rel,
                          const void* workspace, size_t workspace_bytes, void* stream) {
  if (!ctx || !probs || !rel || !workspace) return LEGS_ERR_NULL;
  if (!legs_aligned16(probs) || !legs_aligned16(rel) || !legs_aligned16(workspace)) return LEGS_ERR_ALIGN;
  if ((K != 32 && K != 64 && K != 128) || Q < 1 || Q > kRelQPad || P < 0) return LEGS_ERR_DIM;
  if (workspace_bytes < legs_relevancy_workspace_bytes(K, Q)) return LEGS_ERR_WORKSPACE;
  if (P == 0) return LEGS_OK;
  cudaStream_t st = (cudaStream_t)stream;
  RelParams rp;
  rp.P = P; rp.num_tiles = (P + kRows - 1) / kRows; rp.K = K; rp.Q = Q;
  rp.probs = probs; rp.units = (const uint8_t*)workspace; rp.rel = rel;
  CUtensorMap tmap;
  int rc;
  if ((rc = make_tmap_bf16_2d(ctx, probs, (uint64_t)K, (uint64_t)P, 64, kRows, &tmap)) != LEGS_OK) return rc;
  const int kbs = (K + 63) / 64;
  const int smem_bytes = (2 + kRelStages) * kbs * kUnitBytes + 256 + 1024;
  LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(relevancy_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
  const int grid = (int)(rp.num_tiles < ctx->num_sms ? rp.num_tiles : ctx->num_sms);
  relevancy_kernel<<<grid, kRelThreads, smem_bytes, st>>>(rp, tmap);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

int legs_relevancy(legs_ctx* ctx, const uint16_t* probs, int64_t P, const uint16_t* codebook, int32_t K, int32_t d,
                   int32_t d_clip, const uint16_t* queries, int32_t Q, float* rel, void* workspace,
                   size_t workspace_bytes, void* stream) {
  if (!ctx || !probs || !rel) return LEGS_ERR_NULL;
  if (!legs_aligned16(probs) || !legs_aligned16(rel)) return LEGS_ERR_ALIGN;
  if (P < 0) return LEGS_ERR_DIM;
  int rc;
  if ((rc = legs_relevancy_prepare(ctx, codebook, K, d, d_clip, queries, Q, workspace, workspace_bytes, stream)) != LEGS_OK) return rc;
  return legs_relevancy_packed(ctx, probs, P, K, Q, rel, workspace, workspace_bytes, stream);
}

}  // extern "C"

// =========================================================================================================
// legs_relevancy_static: legs_relevancy for callers that cannot give the library any scratch memory.
//
// Who that is: code that runs where device allocation is forbidden or impossible — a render / serving loop that took all
// of its memory from a pool at start-up and must not touch cudaMalloc afterwards (an allocation may synchronise the whole
// device and stall every other stream), a plugin that is handed input and output buffers by a host application and owns no
// allocator, or a process whose memory budget is already fully committed. legs_relevancy needs 32-64 KB for the packed
// Gram matrix S_c S_c^T and the projected queries S_c q / |q|; every other entry point leaves that to the caller, this
// one keeps it in the array below, which lives in the library's own device image.
//
// The array costs kRelStaticBytes (64 KB) on every GPU that loads liblegs.so, from load until the process exits, whether
// or not this entry point is ever called. In host code `g_rel_static_scratch` is only a handle for the runtime, not an
// address a kernel may be given; the device address is asked for once per device (rel_static_scratch_address) and cached.
namespace {

constexpr int kRelStaticMaxK = 128;                                                     // codes (rows of the codebook)
constexpr size_t kRelStaticBytes = (size_t)2 * ((kRelStaticMaxK + 63) / 64) * kUnitBytes;  // 64 KB: G and V units
static __device__ __align__(256) uint8_t g_rel_static_scratch[kRelStaticBytes];

constexpr int kRelStaticMaxDevices = 64;
std::mutex g_rel_static_mutex;
void* g_rel_static_addr[kRelStaticMaxDevices];  // device address of the array on each device, 0 = not asked for yet

// Device address of the scratch array on ctx's device. The address belongs to the device that is current when it is asked
// for, so the caller's current device must be the context's; the first call per device does the look-up.
int rel_static_scratch_address(legs_ctx* ctx, void** out) {
  int current = -1;
  LEGS_CUDA_CHECK(ctx, cudaGetDevice(&current));
  if (current != ctx->device || current < 0 || current >= kRelStaticMaxDevices) {
    ctx->last_cuda_error = (int)cudaErrorInvalidDevice;
    return LEGS_ERR_CUDA;
  }
  std::lock_guard<std::mutex> lock(g_rel_static_mutex);
  if (!g_rel_static_addr[current]) {
    void* addr = nullptr;
    LEGS_CUDA_CHECK(ctx, cudaGetSymbolAddress(&addr, g_rel_static_scratch));
    if (!addr || (((uintptr_t)addr) & 255u)) {
      ctx->last_cuda_error = (int)cudaErrorInvalidSymbol;
      return LEGS_ERR_CUDA;
    }
    g_rel_static_addr[current] = addr;
  }
  *out = g_rel_static_addr[current];
  return LEGS_OK;
}

}  // namespace

extern "C" {

size_t legs_relevancy_static_bytes(void) { return kRelStaticBytes; }
int32_t legs_relevancy_static_max_codes(void) { return kRelStaticMaxK; }

int legs_relevancy_static(legs_ctx* ctx, const uint16_t* probs, int64_t P, const uint16_t* codebook, int32_t K, int32_t d,
                          int32_t d_clip, const uint16_t* queries, int32_t Q, float* rel, void* stream) {
  if (!ctx || !probs || !rel || !codebook || !queries) return LEGS_ERR_NULL;
  if (!legs_aligned16(probs) || !legs_aligned16(rel) || !legs_aligned16(codebook) || !legs_aligned16(queries)) return LEGS_ERR_ALIGN;
  // sizes the fixed array cannot hold (or the kernels do not take) are refused before anything is enqueued
  if (K > kRelStaticMaxK || legs_relevancy_workspace_bytes(K, Q) > kRelStaticBytes) return LEGS_ERR_DIM;
  if (P < 0) return LEGS_ERR_DIM;
  void* scratch = nullptr;
  int rc;
  if ((rc = rel_static_scratch_address(ctx, &scratch)) != LEGS_OK) return rc;
  // From here on it is the two-step path of legs_relevancy on the library's own memory. legs_relevancy_prepare clears the
  // part of the array it uses (the array still holds the previous call's Gram matrix) and repacks it.
  if ((rc = legs_relevancy_prepare(ctx, codebook, K, d, d_clip, queries, Q, scratch, kRelStaticBytes, stream)) != LEGS_OK) return rc;
  return legs_relevancy_packed(ctx, probs, P, K, Q, rel, scratch, kRelStaticBytes, stream);
}

}  // extern "C"

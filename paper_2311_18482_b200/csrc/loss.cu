// loss.cu — semantic loss head (Eq. 8-12), forward and reverse mode in one
// persistent tcgen05 kernel:
//   h = relu(W0 x + b0)        (fp32 pipes; in_dim is 8 or 16)
//   z = W1 h + b1              (UMMA: A = h tile, K-major)
//   CE = logsumexp(z) - z[m];  L_CE += CE (1 - u) / P;  L_u += u / P;  dz = lambda_ce (1 - u) / P (softmax(z) - onehot(m))
//   dh = dz W1                 (UMMA: A = dz tile, K-major over the codes)
//   dW1 += dz^T h, db1 += dz^T 1   (UMMA: the SAME dz and h tiles read MN-major: contraction over the 128 pixels;
//                                   accumulated in TMEM over all tiles of the CTA)
//   dpre = dh [pre > 0];  dx = W0^T dpre (fp32 pipes);  dW0 += dpre^T x, db0 += dpre^T 1 (UMMA, MN-major, in TMEM)
// TWO persistent CTAs per SM (104 KB of shared memory, 256 TMEM columns and at most 112 registers each): a tile is a chain of
// three row-thread / MMA hand-offs, so one CTA alone leaves the SM idle most of the time; the second fills the gaps.
// 128-pixel tiles. Warp 0 issues the MMAs; warps 1-8 are 256 row threads (two per pixel, splitting the columns of every
// step). dh reads the SAME W1 tile as the logits (MN-major view: no transposed copy) and lands in the TMEM columns the
// logits have left. The softmax re-reads the logits from TMEM (max / sum / dz passes) instead of holding 64 of them in
// registers. The weight gradients leave TMEM once, at the end, through fp32 atomics.
#include <string.h>

#include "common.cuh"
#include "tc05.cuh"

// 3-layer (Table 3) decoders: loss3.cu
size_t legs_loss3_workspace_bytes(int64_t P);
int legs_loss3_check(const legs_decoder* dec, int sem_dim);
int legs_loss3_launch(legs_ctx* ctx, const float* pixels, int64_t P, int32_t sem_dim, const int32_t* index_map,
                      const legs_decoder* dec, float lambda_ce, float lambda_u, float* dL_dpixels, const legs_decoder_grads* grads,
                      float* loss, void* workspace, cudaStream_t st);

namespace {

using namespace tc05;

constexpr int kRows = 128;
constexpr int kUnit = 16384;            // [128 rows][64 bf16], 128-byte swizzle
constexpr int kRowWarps = 8;
constexpr int kLossThreads = 32 * (1 + kRowWarps);
// shared-memory units
constexpr int kUH = 0, kUDz = 1 /* 2 units */, kUDpre = 3, kUX = 4, kUW1 = 5, kUnits = 6;
// TMEM columns
constexpr int kCZ = 0, kCDh = 0 /* over the logits, once the row threads have read them */, kCDW1 = 128, kCDb1 = 192, kCDW0 = 224, kCols = 256;

struct LossParams {
  long long P, num_tiles;
  int F, CH, h0, K;
  const float* pixels;
  const int* index;
  const uint8_t* units;   // packed: W1 (one B unit)
  const float* consts;    // W0 [h0][F] fp32, b0 [h0], b1 [K]
  float lambda_ce, lambda_u;
  float* dL;
  float *dw0, *db0, *dw1, *db1;
  float* loss;
};

__device__ __forceinline__ float bf16f(uint16_t v) { return __uint_as_float((uint32_t)v << 16); }

// weights -> B units + fp32 constants
__global__ void __launch_bounds__(256) loss_pack_kernel(const uint16_t* __restrict__ w0, const float* __restrict__ b0,
                                                        const uint16_t* __restrict__ w1, const float* __restrict__ b1, int F,
                                                        int h0, int K, uint8_t* units, float* consts) {
  const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
  // one unit: B[n = code][k = hidden] = W1[n][k] (K-major for the logits; read MN-major, k = code, for dh = dz W1)
  for (int c = tid; c < kUnit / 16; c += nth) {
    const int r = c / 8, ch = c % 8;
    uint16_t v[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      const int k = ch * 8 + e;
      v[e] = (r < K && k < h0) ? w1[(size_t)r * h0 + k] : (uint16_t)0;
    }
    uint4 q;
    q.x = v[0] | ((uint32_t)v[1] << 16); q.y = v[2] | ((uint32_t)v[3] << 16);
    q.z = v[4] | ((uint32_t)v[5] << 16); q.w = v[6] | ((uint32_t)v[7] << 16);
    *reinterpret_cast<uint4*>(units + sw128_offset((uint32_t)r, (uint32_t)ch)) = q;
  }
  for (int i = tid; i < h0 * F; i += nth) consts[i] = bf16f(w0[i]);
  for (int i = tid; i < h0; i += nth) consts[h0 * F + i] = b0 ? b0[i] : 0.f;
  for (int i = tid; i < K; i += nth) consts[h0 * F + h0 + i] = b1 ? b1[i] : 0.f;
}

struct LossBarriers {
  uint64_t a_ready, z_ready, dz_ready, g_ready, dpre_ready, tile_done;
  uint32_t tmem_base;
};

constexpr int kOffConsts = kUnits * kUnit;                       // fp32 constants (<= 64*16 + 64 + 128 floats)
constexpr int kOffXch = kOffConsts + 5120;                       // pair exchange: [2][128] max, [2][128] sum, [2][128] zm
constexpr int kOffBars = kOffXch + 6 * 128 * 4;
constexpr int kLossSmem = kOffBars + 256;                        // 104.5 KB: two CTAs per SM

// pair exchange of dx (up to 16 floats per row) in the logical chunks 4..7 of the x tile's rows (the MMAs read chunks 0..3)
__device__ __forceinline__ float* dx_slot(uint8_t* t_x, int row, int f) {
  return reinterpret_cast<float*>(t_x + sw128_offset((uint32_t)row, (uint32_t)(4 + (f >> 2)))) + (f & 3);
}

template <int F>
__global__ void __launch_bounds__(kLossThreads, 2) loss_kernel(const __grid_constant__ LossParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  float* s_consts = reinterpret_cast<float*>(smem + kOffConsts);
  float* s_xch = reinterpret_cast<float*>(smem + kOffXch);
  LossBarriers* bar = reinterpret_cast<LossBarriers*>(smem + kOffBars);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int h0 = p.h0, K = p.K, CH = p.CH;
  const long long my_tiles = (p.num_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x;

  if (threadIdx.x == 0) {
    mbar_init(&bar->a_ready, kRowWarps * 32); mbar_init(&bar->z_ready, 1);
    mbar_init(&bar->dz_ready, kRowWarps * 32); mbar_init(&bar->g_ready, 1);
    mbar_init(&bar->dpre_ready, kRowWarps * 32); mbar_init(&bar->tile_done, 1);
    fence_barrier_init();
  }
  if (warp == 0) { tmem_alloc(&bar->tmem_base, kCols); tmem_relinquish(); }
  // zero the operand tiles (padding columns stay zero for the whole kernel), load the resident B units and constants
  for (int i = threadIdx.x; i < kUW1 * (kUnit / 16); i += kLossThreads) reinterpret_cast<uint4*>(smem)[i] = make_uint4(0, 0, 0, 0);
  for (int i = threadIdx.x; i < kUnit / 16; i += kLossThreads)
    reinterpret_cast<uint4*>(smem + kUW1 * kUnit)[i] = reinterpret_cast<const uint4*>(p.units)[i];
  for (int i = threadIdx.x; i < h0 * F + h0 + K; i += kLossThreads) s_consts[i] = p.consts[i];
  __syncthreads();
  // the ones column of the x tile (column F): db0 and db1 come out of the same MMAs as dW0 (and a by-product of dz^T x)
  if (threadIdx.x < kRows) {
    const int r = threadIdx.x, chunk = F >> 3;
    *reinterpret_cast<uint16_t*>(smem + kUX * kUnit + sw128_offset(r, chunk) + (F & 7) * 2) = 0x3f80;  // bf16 1.0
  }
  fence_proxy_async_smem();
  fence_before_sync();
  __syncthreads();
  fence_after_sync();
  const uint32_t tmem = bar->tmem_base;

  if (warp == 0) {
    // ===================== MMA issuer (warp-uniform loop, one elected lane issues) =====================
    const uint32_t hiK = kDescHiSw128;                    // K-major: SBO = 1024
    const uint32_t hiMN = desc_hi_sw128(1024);            // MN-major: 8-row (8 k) groups 1024 B apart
    const uint32_t base = smem_u32(smem);
    const uint32_t h_lo = desc_lo(base + kUH * kUnit, 16), dz_lo = desc_lo(base + kUDz * kUnit, 16);
    const uint32_t w1_lo = desc_lo(base + kUW1 * kUnit, 16);
    const uint32_t w1T_lo = desc_lo(base + kUW1 * kUnit, kUnit);   // the same tile, MN-major: k = code (rows), n = hidden
    // MN-major views: LBO = 16 KB between 64-wide M/N groups (dz: codes 0-63 / 64-127; dpre: hidden / the x unit that
    // follows it: rows 64-127 of the dW0 accumulator are never read)
    const uint32_t dzT_lo = desc_lo(base + kUDz * kUnit, kUnit), hT_lo = desc_lo(base + kUH * kUnit, kUnit);
    const uint32_t dpT_lo = desc_lo(base + kUDpre * kUnit, kUnit), xT_lo = desc_lo(base + kUX * kUnit, kUnit);
    const uint32_t id_z = make_idesc_bf16(kRows, (uint32_t)K), id_dh = make_idesc_bf16_major(kRows, 64, 0, 1);
    const uint32_t id_w1 = make_idesc_bf16_major(128, 64, 1, 1), id_b = make_idesc_bf16_major(128, 32, 1, 1);
    uint32_t par = 0;
    for (long long i = 0; i < my_tiles; ++i, par ^= 1) {
      const uint32_t acc = i > 0 ? 1u : 0u;
      mbar_wait(&bar->a_ready, par);
      fence_after_sync();
      if (elect_one_sync()) {
        for (int k = 0; k < h0 / 16; ++k) umma_bf16_desc(tmem + kCZ, h_lo + 2 * k, hiK, w1_lo + 2 * k, hiK, id_z, k ? 1u : 0u);
        umma_commit(&bar->z_ready);
      }
      __syncwarp();
      mbar_wait(&bar->dz_ready, par);
      fence_after_sync();
      if (elect_one_sync()) {
        for (int k = 0; k < K / 16; ++k) {   // dh = dz W1: contraction over the codes (A: 64 per k-block unit; B: 16 rows per step)
          const uint32_t off = (k >> 2) * (kUnit >> 4) + 2 * (k & 3);
          umma_bf16_desc(tmem + kCDh, dz_lo + off, hiK, w1T_lo + (uint32_t)k * (2048u >> 4), hiMN, id_dh, k ? 1u : 0u);
        }
        umma_commit(&bar->g_ready);              // the row threads only wait for dh; the weight gradients follow
        for (int k = 0; k < kRows / 16; ++k) {   // contraction over the pixels: 16 rows = 2048 B per step
          const uint32_t off = k * (2048 >> 4);
          umma_bf16_desc(tmem + kCDW1, dzT_lo + off, hiMN, hT_lo + off, hiMN, id_w1, acc | (k ? 1u : 0u));
          umma_bf16_desc(tmem + kCDb1, dzT_lo + off, hiMN, xT_lo + off, hiMN, id_b, acc | (k ? 1u : 0u));
        }
      }
      __syncwarp();
      mbar_wait(&bar->dpre_ready, par);
      fence_after_sync();
      if (elect_one_sync()) {
        for (int k = 0; k < kRows / 16; ++k) {
          const uint32_t off = k * (2048 >> 4);
          umma_bf16_desc(tmem + kCDW0, dpT_lo + off, hiMN, xT_lo + off, hiMN, id_b, acc | (k ? 1u : 0u));
        }
        umma_commit(&bar->tile_done);
      }
      __syncwarp();
    }
  } else {
    // ===================== 256 row threads: pixel row = TMEM lane, two threads per row split the columns ===========
    const int row = 32 * (warp & 3) + lane;
    const int hf = (warp - 1) >> 2;
    const uint32_t lane_addr = tmem + ((uint32_t)(32 * (warp & 3)) << 16);
    uint8_t* a_h = smem + kUH * kUnit;
    uint8_t* a_dz = smem + kUDz * kUnit;
    uint8_t* a_dp = smem + kUDpre * kUnit;
    uint8_t* a_x = smem + kUX * kUnit;
    const float* W0 = s_consts;
    const float* b0 = s_consts + h0 * F;
    const float* b1 = b0 + h0;
    float* x_max = s_xch;              // [2][128]
    float* x_sum = s_xch + 256;        // [2][128]
    float* x_zm = s_xch + 512;         // [2][128]
    const float invP = 1.0f / (float)p.P;
    float acc_ce = 0.f, acc_u = 0.f;
    uint32_t par = 0;
    const int nch = h0 / 8;            // 16-byte chunks of the hidden layer; this thread owns chunks hf, hf + 2, ...
    float nx[F], nu = 1.f;
    int nm = 0;
    auto fetch = [&](long long t) {
      const long long r = t * kRows + row;
#pragma unroll
      for (int k = 0; k < F; ++k) nx[k] = 0.f;
      nu = 1.f; nm = 0;
      if (r < p.P) {
        const float4* px = reinterpret_cast<const float4*>(p.pixels + r * CH + 4);
        float v[F + 4];
#pragma unroll
        for (int k = 0; k < F / 4 + 1; ++k) { const float4 q = px[k]; v[4 * k] = q.x; v[4 * k + 1] = q.y; v[4 * k + 2] = q.z; v[4 * k + 3] = q.w; }
#pragma unroll
        for (int k = 0; k < F; ++k) nx[k] = v[k];
        nu = v[F];
        nm = p.index[r];
      }
    };
    fetch(blockIdx.x);
    for (long long i = 0; i < my_tiles; ++i, par ^= 1) {
      const long long tile = blockIdx.x + i * gridDim.x;
      const long long prow = tile * kRows + row;
      const bool valid = prow < p.P;
      // ---- F1: pixel row (fetched one tile ahead), layer 0
      float x[F];
#pragma unroll
      for (int k = 0; k < F; ++k) x[k] = nx[k];
      const float u = nu;
      const int m = nm;
      uint32_t relu_mask = 0;          // bit (own chunk index * 8 + e)
      uint4 hq[4];
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        const int c = hf + 2 * t;
        hq[t] = make_uint4(0, 0, 0, 0);
        if (c < nch) {
          float h[8];
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            const float4* wr = reinterpret_cast<const float4*>(W0 + (c * 8 + e) * F);
            float a = b0[c * 8 + e];
#pragma unroll
            for (int k = 0; k < F / 4; ++k) {
              const float4 w = wr[k];
              a = fmaf(w.x, x[4 * k], a); a = fmaf(w.y, x[4 * k + 1], a); a = fmaf(w.z, x[4 * k + 2], a); a = fmaf(w.w, x[4 * k + 3], a);
            }
            if (a > 0.f) relu_mask |= 1u << (t * 8 + e);
            h[e] = fmaxf(a, 0.f);
          }
          hq[t] = make_uint4(pack_bf16(h[0], h[1]), pack_bf16(h[2], h[3]), pack_bf16(h[4], h[5]), pack_bf16(h[6], h[7]));
        }
      }
      if (i > 0) { mbar_wait(&bar->tile_done, par ^ 1); fence_after_sync(); }   // the MMAs of the last tile have read the tiles
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        const int c = hf + 2 * t;
        if (c < nch) *reinterpret_cast<uint4*>(a_h + sw128_offset(row, c)) = hq[t];
      }
      if (hf == 0) {
        const uint4 q0 = make_uint4(pack_bf16(x[0], x[1]), pack_bf16(x[2], x[3]), pack_bf16(x[4], x[5]), pack_bf16(x[6], x[7]));
        *reinterpret_cast<uint4*>(a_x + sw128_offset(row, 0)) = q0;
        if constexpr (F == 16) {
          const uint4 q1 = make_uint4(pack_bf16(x[8], x[9]), pack_bf16(x[10], x[11]), pack_bf16(x[12], x[13]), pack_bf16(x[14], x[15]));
          *reinterpret_cast<uint4*>(a_x + sw128_offset(row, 1)) = q1;
        }
      }
      fence_proxy_async_smem();
      mbar_arrive(&bar->a_ready);
      if (i + 1 < my_tiles) fetch(tile + gridDim.x);
      // ---- F2: softmax, cross entropy, dz
      mbar_wait(&bar->z_ready, par);
      fence_after_sync();
      // three passes over this thread's logits in TMEM (max and z[m]; sum of exponentials; dz): 32 live values at a time
      const int ng = K / 32;
      float mx = -3.0e38f, zm = 0.f;
#pragma unroll
      for (int t = 0; t < 2; ++t) {
        const int g = hf + 2 * t;
        if (g < ng) {
          uint32_t r[32];
          tmem_ld32(lane_addr + kCZ + g * 32, r);
          tmem_ld_wait();
#pragma unroll
          for (int e = 0; e < 32; ++e) {
            const float zv = __uint_as_float(r[e]) + b1[g * 32 + e];
            mx = fmaxf(mx, zv);
            if (g * 32 + e == m) zm = zv;
          }
        }
      }
      x_max[hf * kRows + row] = mx;
      x_zm[hf * kRows + row] = zm;
      asm volatile("bar.sync 1, %0;" ::"n"(kRowWarps * 32) : "memory");
      mx = fmaxf(mx, x_max[(hf ^ 1) * kRows + row]);
      zm += x_zm[(hf ^ 1) * kRows + row];
      float sum = 0.f;
#pragma unroll
      for (int t = 0; t < 2; ++t) {
        const int g = hf + 2 * t;
        if (g < ng) {
          uint32_t r[32];
          tmem_ld32(lane_addr + kCZ + g * 32, r);
          tmem_ld_wait();
#pragma unroll
          for (int e = 0; e < 32; ++e) sum += __expf((__uint_as_float(r[e]) + b1[g * 32 + e]) - mx);
        }
      }
      x_sum[hf * kRows + row] = sum;
      asm volatile("bar.sync 1, %0;" ::"n"(kRowWarps * 32) : "memory");
      sum += x_sum[(hf ^ 1) * kRows + row];
      const float ce = (mx + __logf(sum)) - zm;
      const float coef = valid ? p.lambda_ce * (1.0f - u) * invP : 0.f;
      const float scale = coef / sum;
#pragma unroll
      for (int t = 0; t < 2; ++t) {
        const int g = hf + 2 * t;
        if (g < ng) {
          uint32_t r[32];
          tmem_ld32(lane_addr + kCZ + g * 32, r);
          tmem_ld_wait();
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            float d[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) {
              const int code = g * 32 + c * 8 + e;
              d[e] = __expf((__uint_as_float(r[c * 8 + e]) + b1[code]) - mx) * scale - ((code == m) ? coef : 0.f);
            }
            const uint4 q = make_uint4(pack_bf16(d[0], d[1]), pack_bf16(d[2], d[3]), pack_bf16(d[4], d[5]), pack_bf16(d[6], d[7]));
            const int chunk = g * 4 + c;
            *reinterpret_cast<uint4*>(a_dz + (chunk >> 3) * kUnit + sw128_offset(row, chunk & 7)) = q;
          }
        }
      }
      fence_before_sync();   // the logits have been read for the last time: dh may overwrite their columns
      if (hf == 0 && valid) {
        acc_ce += ce * (1.0f - u);
        acc_u += u;
        p.dL[prow * CH + 4 + F] = (p.lambda_u - p.lambda_ce * ce) * invP;
      }
      fence_proxy_async_smem();
      mbar_arrive(&bar->dz_ready);
      // ---- F3: dpre = dh [pre > 0], dx = W0^T dpre
      mbar_wait(&bar->g_ready, par);
      fence_after_sync();
      float dx[F];
#pragma unroll
      for (int k = 0; k < F; ++k) dx[k] = 0.f;
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        const int c = hf + 2 * t;
        if (c < nch) {
          uint32_t r[8];
          tmem_ld8(lane_addr + kCDh + c * 8, r);
          tmem_ld_wait();
          float d[8];
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            d[e] = ((relu_mask >> (t * 8 + e)) & 1u) ? __uint_as_float(r[e]) : 0.f;
            const float4* wr = reinterpret_cast<const float4*>(W0 + (c * 8 + e) * F);
#pragma unroll
            for (int k = 0; k < F / 4; ++k) {
              const float4 w = wr[k];
              dx[4 * k] = fmaf(w.x, d[e], dx[4 * k]); dx[4 * k + 1] = fmaf(w.y, d[e], dx[4 * k + 1]);
              dx[4 * k + 2] = fmaf(w.z, d[e], dx[4 * k + 2]); dx[4 * k + 3] = fmaf(w.w, d[e], dx[4 * k + 3]);
            }
          }
          *reinterpret_cast<uint4*>(a_dp + sw128_offset(row, c)) =
              make_uint4(pack_bf16(d[0], d[1]), pack_bf16(d[2], d[3]), pack_bf16(d[4], d[5]), pack_bf16(d[6], d[7]));
        }
      }
      fence_before_sync();
      fence_proxy_async_smem();
      mbar_arrive(&bar->dpre_ready);
      if (hf == 1) {
#pragma unroll
        for (int k = 0; k < F; ++k) *dx_slot(a_x, row, k) = dx[k];
      }
      asm volatile("bar.sync 1, %0;" ::"n"(kRowWarps * 32) : "memory");
      if (hf == 0 && valid) {
        float* o = p.dL + prow * CH + 4;
#pragma unroll
        for (int k = 0; k < F; k += 4)
          *reinterpret_cast<float4*>(o + k) = make_float4(dx[k] + *dx_slot(a_x, row, k), dx[k + 1] + *dx_slot(a_x, row, k + 1),
                                                          dx[k + 2] + *dx_slot(a_x, row, k + 2), dx[k + 3] + *dx_slot(a_x, row, k + 3));
      }
    }
    // ---- end of the CTA's tiles: weight gradients leave TMEM (lane = code or hidden unit), losses are reduced
    mbar_wait(&bar->tile_done, par ^ 1);
    fence_after_sync();
    {
      // dW1 [K][h0]: lane = code, columns kCDW1 + hidden; this thread takes hidden [hf*32, hf*32 + 32)
      uint32_t r[32];
      tmem_ld32(lane_addr + kCDW1 + hf * 32, r);
      tmem_ld_wait();
      if (row < K) {
#pragma unroll
        for (int e = 0; e < 32; ++e) {
          const int j = hf * 32 + e;
          if (j < h0) atomicAdd(p.dw1 + (size_t)row * h0 + j, __uint_as_float(r[e]));
        }
      }
      if (hf == 0) {
        // db1: column F of the dz^T [x | 1] product; dW0 / db0: rows = hidden units, columns = inputs | 1
        tmem_ld32(lane_addr + kCDb1, r);
        tmem_ld_wait();
        if (row < K && p.db1) atomicAdd(p.db1 + row, __uint_as_float(r[F]));
        tmem_ld32(lane_addr + kCDW0, r);
        tmem_ld_wait();
        if (row < h0) {
#pragma unroll
          for (int e = 0; e < F; ++e) atomicAdd(p.dw0 + (size_t)row * F + e, __uint_as_float(r[e]));
          if (p.db0) atomicAdd(p.db0 + row, __uint_as_float(r[F]));
        }
      }
    }
    fence_before_sync();
    for (int o = 16; o > 0; o >>= 1) { acc_ce += __shfl_xor_sync(0xffffffffu, acc_ce, o); acc_u += __shfl_xor_sync(0xffffffffu, acc_u, o); }
    if (lane == 0 && hf == 0) {
      const float lce = acc_ce * invP, lu = acc_u * invP;
      atomicAdd(p.loss + 0, lce);
      atomicAdd(p.loss + 1, lu);
      atomicAdd(p.loss + 2, p.lambda_ce * lce + p.lambda_u * lu);
    }
  }
  fence_before_sync();
  __syncthreads();
  if (warp == 0) { fence_after_sync(); tmem_dealloc(tmem, kCols); }
}

int check_loss_decoder(const legs_decoder* dec, int sem_dim) {
  if (!dec) return LEGS_ERR_NULL;
  if (dec->n_layers != 2 && dec->n_layers != 3) return LEGS_ERR_DIM;
  if (dec->n_layers == 3) {
    const int rc = legs_loss3_check(dec, sem_dim);
    if (rc != LEGS_OK) return rc;
  } else {
    if ((sem_dim != 8 && sem_dim != 16) || dec->in_dim != sem_dim) return LEGS_ERR_DIM;
    if (dec->hidden[0] != 32 && dec->hidden[0] != 64) return LEGS_ERR_DIM;
    if (dec->n_codes != 32 && dec->n_codes != 64 && dec->n_codes != 128) return LEGS_ERR_DIM;
  }
  for (int l = 0; l < dec->n_layers; ++l) {
    if (!dec->w[l]) return LEGS_ERR_NULL;
    if (!legs_aligned16(dec->w[l]) || (dec->b[l] && !legs_aligned16(dec->b[l]))) return LEGS_ERR_ALIGN;
  }
  return LEGS_OK;
}

}  // namespace

extern "C" {

size_t legs_loss_workspace_bytes(const legs_decoder* dec, int64_t P) {
  if (dec && dec->n_layers == 3) return legs_loss3_workspace_bytes(P < 0 ? 0 : P);
  return (size_t)kUnit + 8192;
}

int legs_semantic_loss(legs_ctx* ctx, const float* pixels, int64_t P, int32_t sem_dim, const int32_t* index_map,
                       const legs_decoder* dec, float lambda_ce, float lambda_u, float* dL_dpixels,
                       const legs_decoder_grads* grads, float* loss, void* workspace, size_t workspace_bytes, void* stream) {
  if (!ctx) return LEGS_ERR_NULL;
  int rc;
  if ((rc = check_loss_decoder(dec, sem_dim)) != LEGS_OK) return rc;
  if (!pixels || !index_map || !dL_dpixels || !grads || !loss || !workspace) return LEGS_ERR_NULL;
  for (int l = 0; l < dec->n_layers; ++l) {
    if (!grads->dw[l]) return LEGS_ERR_NULL;
    if (!legs_aligned16(grads->dw[l]) || (grads->db[l] && !legs_aligned16(grads->db[l]))) return LEGS_ERR_ALIGN;
  }
  if (!legs_aligned16(pixels) || !legs_aligned16(index_map) || !legs_aligned16(dL_dpixels) || !legs_aligned16(loss) ||
      !legs_aligned16(workspace))
    return LEGS_ERR_ALIGN;
  if (P < 0) return LEGS_ERR_DIM;
  if (workspace_bytes < legs_loss_workspace_bytes(dec, P)) return LEGS_ERR_WORKSPACE;
  if (P == 0) return LEGS_OK;
  cudaStream_t st = (cudaStream_t)stream;
  if (dec->n_layers == 3)
    return legs_loss3_launch(ctx, pixels, P, sem_dim, index_map, dec, lambda_ce, lambda_u, dL_dpixels, grads, loss, workspace, st);
  uint8_t* units = (uint8_t*)workspace;
  float* consts = (float*)(units + kUnit);
  loss_pack_kernel<<<16, 256, 0, st>>>(dec->w[0], dec->b[0], dec->w[1], dec->b[1], sem_dim, dec->hidden[0], dec->n_codes, units,
                                       consts);
  LEGS_LAUNCH_CHECK(ctx);
  LossParams lp;
  lp.P = P; lp.num_tiles = (P + kRows - 1) / kRows;
  lp.F = sem_dim; lp.CH = legs_pixel_channels(sem_dim); lp.h0 = dec->hidden[0]; lp.K = dec->n_codes;
  lp.pixels = pixels; lp.index = index_map; lp.units = units; lp.consts = consts;
  lp.lambda_ce = lambda_ce; lp.lambda_u = lambda_u; lp.dL = dL_dpixels;
  lp.dw0 = grads->dw[0]; lp.db0 = grads->db[0]; lp.dw1 = grads->dw[1]; lp.db1 = grads->db[1];
  lp.loss = loss;
  const int smem_bytes = kLossSmem + 1024;
  const long long slots = 2ll * ctx->num_sms;   // two CTAs per SM
  const int grid = (int)(lp.num_tiles < slots ? lp.num_tiles : slots);
  if (sem_dim == 8) {
    LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(loss_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
    loss_kernel<8><<<grid, kLossThreads, smem_bytes, st>>>(lp);
  } else {
    LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(loss_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
    loss_kernel<16><<<grid, kLossThreads, smem_bytes, st>>>(lp);
  }
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

}  // extern "C"

// loss3.cu — semantic loss head (Eq. 8-12) for the paper's own decoder,
// Table 3: F -> 128 -> 256 -> K, forward and reverse mode.
//   h0 = relu(W0 x + b0)          (fp32 pipes; F = 8 or 16)
//   h1 = relu(W1 h0 + b1)         (UMMA, N = 256 taken as 128 + 64 + 64 columns through two scratch accumulators)
//   z  = W2 h1 + b2               (UMMA, K = 256)
//   CE, L_CE, L_u, dz             (fp32 pipes, as in loss.cu)
//   dh1 = dz W2   (UMMA; B = the SAME W2 tile read MN-major),  dpre1 = dh1 [pre1 > 0]
//   dW2 += dz^T h1, db2 += dz^T 1 (UMMA over MN-major views: contraction over the tile's 128 pixels, accumulated in
//                                  TMEM over all tiles of the CTA)
//   dh0 = dpre1 W1 (UMMA; B = W1 read MN-major),  dpre0 = dh0 [pre0 > 0],  dx = W0^T dpre0 (fp32 pipes)
//   dW0 += dpre0^T x, db0 += dpre0^T 1 (UMMA, in TMEM)
// dW2 [K x 256] and dW1 [256 x 128] are 256 TMEM columns each: together they would leave no scratch accumulator, and the
// two weight tiles (64 KB each) do not fit beside the activation tiles either. So:
//   * W1 and W2 take turns in ONE 64 KB shared-memory buffer, streamed from L2 by bulk async copies twice per tile;
//   * loss3_kernel keeps dW2 (+ db2, dW0, db0) in TMEM and saves the operands of dW1 — the h0 and dpre1 tiles, exactly as
//     they sit in shared memory (bf16, 128-byte swizzle) — to the workspace with bulk stores (768 B per pixel);
//   * loss3_dw1_kernel streams those tiles back (two-stage ring of bulk copies) and accumulates dW1 += dpre1^T h0 and
//     db1 += dpre1^T 1 in TMEM: no row threads, no hand-offs.
#include "common.cuh"
#include "tc05.cuh"

namespace {

using namespace tc05;

constexpr int kRows = 128;
constexpr int kH0 = 128, kH1 = 256;
constexpr int kUnit = 16384;            // [128 rows][64 bf16], 128-byte swizzle
constexpr uint32_t kUnitLo = kUnit >> 4;
constexpr int kRowWarps = 8;
constexpr int kThreads = 32 * (1 + kRowWarps);
// shared-memory units of loss3_kernel
constexpr int kUX = 0, kUH0 = 1 /* 2 */, kUH1 = 3 /* 4: h1, then dpre1 */, kUDz = 7 /* 2: dz, then dpre0 */, kUWB = 9 /* 4 */, kUnits = 13;
// TMEM columns of loss3_kernel
constexpr int kCS0 = 0, kCS1 = 128, kCDW2 = 192, kCDb2 = 448, kCDW0 = 480;
// workspace
constexpr size_t kWsW1 = 0, kWsW2 = 65536, kWsConsts = 131072, kWsSave = 131072 + 16384;
constexpr size_t kSaveTile = 6 * (size_t)kUnit;    // h0 (2 units) + dpre1 (4 units) per 128-pixel tile

struct Loss3Params {
  long long P, num_tiles;
  int F, CH, K;
  const float* pixels;
  const int* index;
  const uint8_t* wpack;   // W1 (2 k-block units of [256][64]), W2 (4 k-block units of [128][64])
  const float* consts;    // W0 [128][F] fp32, b0 [128], b1 [256], b2 [128]
  uint8_t* save;
  float lambda_ce, lambda_u;
  float* dL;
  float *dw0, *db0, *dw1, *db1, *dw2, *db2;
  float* loss;
};

__device__ __forceinline__ float bf16f(uint16_t v) { return __uint_as_float((uint32_t)v << 16); }

__device__ __forceinline__ void bulk_s2g(void* dst_gmem, const void* src_smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)), "r"(bytes)
               : "memory");
}

__global__ void __launch_bounds__(256) loss3_pack_kernel(const uint16_t* __restrict__ w0, const float* __restrict__ b0,
                                                         const uint16_t* __restrict__ w1, const float* __restrict__ b1,
                                                         const uint16_t* __restrict__ w2, const float* __restrict__ b2, int F, int K,
                                                         uint8_t* wpack, float* consts) {
  const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
  // W1 [256][128]: B[n = hidden1][k = hidden0], two k-blocks of 64, each [256 rows][64] = 32 KB
  for (int c = tid; c < 2 * kH1 * 8; c += nth) {
    const int kb = c / (kH1 * 8), w = c % (kH1 * 8), n = w / 8, ch = w % 8;
    *reinterpret_cast<uint4*>(wpack + kWsW1 + (size_t)kb * 2 * kUnit + sw128_offset((uint32_t)n, (uint32_t)ch)) =
        *reinterpret_cast<const uint4*>(w1 + (size_t)n * kH0 + kb * 64 + ch * 8);
  }
  // W2 [K][256]: B[n = code][k = hidden1], four k-blocks of 64, each [128 rows][64] = 16 KB (rows >= K are zero)
  for (int c = tid; c < 4 * kRows * 8; c += nth) {
    const int kb = c / (kRows * 8), w = c % (kRows * 8), n = w / 8, ch = w % 8;
    uint4 q = make_uint4(0, 0, 0, 0);
    if (n < K) q = *reinterpret_cast<const uint4*>(w2 + (size_t)n * kH1 + kb * 64 + ch * 8);
    *reinterpret_cast<uint4*>(wpack + kWsW2 + (size_t)kb * kUnit + sw128_offset((uint32_t)n, (uint32_t)ch)) = q;
  }
  float* cb0 = consts + kH0 * F;
  float* cb1 = cb0 + kH0;
  float* cb2 = cb1 + kH1;
  for (int i = tid; i < kH0 * F; i += nth) consts[i] = bf16f(w0[i]);
  for (int i = tid; i < kH0; i += nth) cb0[i] = b0 ? b0[i] : 0.f;
  for (int i = tid; i < kH1; i += nth) cb1[i] = b1 ? b1[i] : 0.f;
  for (int i = tid; i < kRows; i += nth) cb2[i] = (b2 && i < K) ? b2[i] : 0.f;
}

struct Loss3Barriers {
  uint64_t a0_ready, s0_full, s1_full, s0_free, a1_ready, w_ready, dz_ready, w2_done, mma_done, dp1_ready, dp0_ready, tile_done,
      st_done;
  uint32_t tmem_base;
};

constexpr int kOffConsts = kUnits * kUnit;                         // W0 (<= 128*16) + 128 + 256 + 128 floats
constexpr int kConstFloats = kH0 * 16 + kH0 + kH1 + kRows;
constexpr int kOffXch = kOffConsts + kConstFloats * 4;             // [2][128] max, [2][128] sum, [2][128] z[m]
constexpr int kOffBars = kOffXch + 6 * 128 * 4;
constexpr int kLoss3Smem = kOffBars + 128;

// 32 fp32 values -> bf16 -> four 16-byte chunks (4 q .. 4 q + 3) of row `row` of one [128 x 64] unit
__device__ __forceinline__ void store_quarter_row(uint8_t* unit, int row, int q, const float (&v)[32]) {
#pragma unroll
  for (int c = 0; c < 4; ++c)
    *reinterpret_cast<uint4*>(unit + sw128_offset(row, 4 * q + c)) =
        make_uint4(pack_bf16(v[8 * c], v[8 * c + 1]), pack_bf16(v[8 * c + 2], v[8 * c + 3]), pack_bf16(v[8 * c + 4], v[8 * c + 5]),
                   pack_bf16(v[8 * c + 6], v[8 * c + 7]));
}

// pair exchange of dx (16 floats per row) in the logical chunks 4..7 of the x tile's rows (the MMAs read chunks 0..3)
__device__ __forceinline__ float* dx_slot(uint8_t* t_x, int row, int f) {
  return reinterpret_cast<float*>(t_x + sw128_offset((uint32_t)row, (uint32_t)(4 + (f >> 2)))) + (f & 3);
}

template <int F>
__global__ void __launch_bounds__(kThreads, 1) loss3_kernel(const __grid_constant__ Loss3Params p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  float* s_consts = reinterpret_cast<float*>(smem + kOffConsts);
  float* s_xch = reinterpret_cast<float*>(smem + kOffXch);
  Loss3Barriers* bar = reinterpret_cast<Loss3Barriers*>(smem + kOffBars);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int K = p.K, CH = p.CH;
  const long long my_tiles = (p.num_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x;
  constexpr int kNR = kRowWarps * 32;

  if (threadIdx.x == 0) {
    mbar_init(&bar->a0_ready, kNR); mbar_init(&bar->s0_full, 1); mbar_init(&bar->s1_full, 1); mbar_init(&bar->s0_free, kNR);
    mbar_init(&bar->a1_ready, kNR); mbar_init(&bar->w_ready, 1); mbar_init(&bar->dz_ready, kNR); mbar_init(&bar->w2_done, 1);
    mbar_init(&bar->mma_done, 1); mbar_init(&bar->dp1_ready, kNR); mbar_init(&bar->dp0_ready, kNR); mbar_init(&bar->tile_done, 1);
    mbar_init(&bar->st_done, 1);
    fence_barrier_init();
  }
  if (warp == 0) { tmem_alloc(&bar->tmem_base, 512); tmem_relinquish(); }
  // zero the activation tiles (padding columns of the x and dz tiles stay zero / unread), load the constants
  for (int i = threadIdx.x; i < kUWB * (kUnit / 16); i += kThreads) reinterpret_cast<uint4*>(smem)[i] = make_uint4(0, 0, 0, 0);
  for (int i = threadIdx.x; i < kH0 * F + kH0 + kH1 + kRows; i += kThreads) s_consts[i] = p.consts[i];
  __syncthreads();
  if (threadIdx.x < kRows)   // the ones column of the x tile (column F): db2 and db0 come out of the [x | 1] products
    *reinterpret_cast<uint16_t*>(smem + kUX * kUnit + sw128_offset(threadIdx.x, F >> 3) + (F & 7) * 2) = 0x3f80;
  fence_proxy_async_smem();
  fence_before_sync();
  __syncthreads();
  fence_after_sync();
  const uint32_t tmem = bar->tmem_base;

  if (warp == 0) {
    // ===================== MMA issuer, weight loads, tile saves (warp-uniform waits, lane 0 issues) =====================
    const uint32_t hiK = kDescHiSw128;                    // K-major: SBO = 1024
    const uint32_t hiMN = desc_hi_sw128(1024);            // MN-major: 8-row (8 k) groups 1024 B apart
    const uint32_t base = smem_u32(smem);
    const uint32_t h0_lo = desc_lo(base + kUH0 * kUnit, 16), h1_lo = desc_lo(base + kUH1 * kUnit, 16);
    const uint32_t dz_lo = desc_lo(base + kUDz * kUnit, 16), wb_lo = desc_lo(base + kUWB * kUnit, 16);
    // MN-major views; LBO = distance between 64-wide M/N groups
    const uint32_t dzT = desc_lo(base + kUDz * kUnit, kUnit), h1T = desc_lo(base + kUH1 * kUnit, kUnit);
    const uint32_t xT = desc_lo(base + kUX * kUnit, kUnit);
    const uint32_t w2T = desc_lo(base + kUWB * kUnit, kUnit);        // W2: rows = codes (k), 4 groups of 64 hidden1 units
    const uint32_t w1T = desc_lo(base + kUWB * kUnit, 2 * kUnit);    // W1: rows = hidden1 (k), 2 groups of 64 hidden0 units
    const uint32_t id_f128 = make_idesc_bf16(kRows, 128), id_f64 = make_idesc_bf16(kRows, 64), id_z = make_idesc_bf16(kRows, (uint32_t)K);
    const uint32_t id_b128 = make_idesc_bf16_major(kRows, 128, 0, 1), id_b64 = make_idesc_bf16_major(kRows, 64, 0, 1);
    const uint32_t id_dw2 = make_idesc_bf16_major(128, 256, 1, 1), id_side = make_idesc_bf16_major(128, 32, 1, 1);
    auto gemm_kk = [&](uint32_t dcol, uint32_t a_lo, uint32_t b_lo, uint32_t b_unit_lo, int ksteps, uint32_t idesc) {
      for (int k = 0; k < ksteps; ++k) {
        const uint32_t ao = (k >> 2) * kUnitLo + 2 * (k & 3), bo = (k >> 2) * b_unit_lo + 2 * (k & 3);
        umma_bf16_desc(tmem + dcol, a_lo + ao, hiK, b_lo + bo, hiK, idesc, k ? 1u : 0u);
      }
    };
    auto gemm_kmn = [&](uint32_t dcol, uint32_t a_lo, uint32_t bT_lo, int ksteps, uint32_t idesc) {
      for (int k = 0; k < ksteps; ++k) {   // A K-major; B MN-major: 16 k rows = +2048 B per step
        const uint32_t ao = (k >> 2) * kUnitLo + 2 * (k & 3);
        umma_bf16_desc(tmem + dcol, a_lo + ao, hiK, bT_lo + (uint32_t)k * (2048u >> 4), hiMN, idesc, k ? 1u : 0u);
      }
    };
    auto gemm_rows = [&](uint32_t dcol, uint32_t aT, uint32_t bT, uint32_t idesc, uint32_t acc) {
      for (int k = 0; k < kRows / 16; ++k) {   // contraction over the tile's 128 pixels: both operands MN-major
        const uint32_t off = (uint32_t)k * (2048u >> 4);
        umma_bf16_desc(tmem + dcol, aT + off, hiMN, bT + off, hiMN, idesc, acc | (k ? 1u : 0u));
      }
    };
    auto load_weights = [&](const uint8_t* src) {
      mbar_arrive_expect_tx(&bar->w_ready, 4 * kUnit);
      for (int j = 0; j < 4; ++j) bulk_g2s(smem + (kUWB + j) * kUnit, src + (size_t)j * kUnit, kUnit, &bar->w_ready);
    };
    if (lane == 0) load_weights(p.wpack + kWsW1);
    __syncwarp();
    for (long long i = 0; i < my_tiles; ++i) {
      const long long tile = blockIdx.x + i * gridDim.x;
      const uint32_t par = (uint32_t)(i & 1), acc = i > 0 ? 1u : 0u;
      uint8_t* save = p.save + (size_t)tile * kSaveTile;
      mbar_wait(&bar->a0_ready, par);
      fence_after_sync();
      if (i == 0) mbar_wait(&bar->w_ready, 0);
      if (lane == 0) {
        bulk_s2g(save, smem + kUH0 * kUnit, 2 * kUnit);
        bulk_commit();
        gemm_kk(kCS0, h0_lo, wb_lo, 2 * kUnitLo, 8, id_f128);                          // pre1[:, 0:128]
        umma_commit(&bar->s0_full);
        gemm_kk(kCS1, h0_lo, wb_lo + (128u * 128u >> 4), 2 * kUnitLo, 8, id_f64);      // pre1[:, 128:192]
        umma_commit(&bar->s1_full);
      }
      __syncwarp();
      mbar_wait(&bar->s0_free, 0);
      fence_after_sync();
      if (lane == 0) {
        gemm_kk(kCS0, h0_lo, wb_lo + (192u * 128u >> 4), 2 * kUnitLo, 8, id_f64);      // pre1[:, 192:256]
        umma_commit(&bar->s0_full);
        umma_commit(&bar->mma_done);
      }
      __syncwarp();
      mbar_wait(&bar->mma_done, 0);                      // W1 has been read: the buffer takes W2
      if (lane == 0) load_weights(p.wpack + kWsW2);
      __syncwarp();
      mbar_wait(&bar->a1_ready, par);
      fence_after_sync();
      mbar_wait(&bar->w_ready, 1);
      if (lane == 0) {
        gemm_kk(kCS0, h1_lo, wb_lo, kUnitLo, 16, id_z);                                // z = h1 W2^T
        umma_commit(&bar->s0_full);
      }
      __syncwarp();
      mbar_wait(&bar->dz_ready, par);
      fence_after_sync();
      if (lane == 0) {
        gemm_kmn(kCS0, dz_lo, w2T, K / 16, id_b128);                                   // dh1[:, 0:128] = dz W2
        umma_commit(&bar->s0_full);
        gemm_kmn(kCS1, dz_lo, w2T + 2 * kUnitLo, K / 16, id_b64);                      // dh1[:, 128:192]
        umma_commit(&bar->s1_full);
        gemm_rows(kCDW2, dzT, h1T, id_dw2, acc);                                       // dW2 += dz^T h1
        gemm_rows(kCDb2, dzT, xT, id_side, acc);                                       // . | db2 += dz^T [x | 1]
        umma_commit(&bar->w2_done);                                                    // the h1 tile may be overwritten
      }
      __syncwarp();
      mbar_wait(&bar->s0_free, 1);
      fence_after_sync();
      if (lane == 0) {
        gemm_kmn(kCS0, dz_lo, w2T + 3 * kUnitLo, K / 16, id_b64);                      // dh1[:, 192:256]
        umma_commit(&bar->s0_full);
        umma_commit(&bar->mma_done);
      }
      __syncwarp();
      mbar_wait(&bar->mma_done, 1);                      // W2 has been read: the buffer takes W1 (kept for the next tile)
      if (lane == 0) load_weights(p.wpack + kWsW1);
      __syncwarp();
      mbar_wait(&bar->dp1_ready, par);
      fence_after_sync();
      mbar_wait(&bar->w_ready, 0);
      if (lane == 0) {
        bulk_s2g(save + 2 * kUnit, smem + kUH1 * kUnit, 4 * kUnit);
        bulk_commit();
        gemm_kmn(kCS0, h1_lo, w1T, 16, id_b128);                                       // dh0 = dpre1 W1
        umma_commit(&bar->s0_full);
      }
      __syncwarp();
      mbar_wait(&bar->dp0_ready, par);
      fence_after_sync();
      if (lane == 0) {
        gemm_rows(kCDW0, dzT, xT, id_side, acc);                                       // dW0 | db0 += dpre0^T [x | 1]
        umma_commit(&bar->tile_done);
        bulk_wait_read<0>();                                                           // both saves have left shared memory
        mbar_arrive(&bar->st_done);
      }
      __syncwarp();
    }
    if (lane == 0) bulk_wait<0>();
    __syncwarp();
  } else {
    // ===================== 256 row threads: pixel row = TMEM lane, two threads per row split the columns ===========
    const int row = 32 * (warp & 3) + lane;
    const int hf = (warp - 1) >> 2;
    const uint32_t lane_addr = tmem + ((uint32_t)(32 * (warp & 3)) << 16);
    uint8_t* t_x = smem + kUX * kUnit;
    uint8_t* t_h0 = smem + kUH0 * kUnit;
    uint8_t* t_h1 = smem + kUH1 * kUnit;
    uint8_t* t_dz = smem + kUDz * kUnit;
    const float* W0 = s_consts;
    const float* b0 = s_consts + kH0 * F;
    const float* b1 = b0 + kH0;
    const float* b2 = b1 + kH1;
    float* x_max = s_xch;              // [2][128]
    float* x_sum = s_xch + 256;
    float* x_zm = s_xch + 512;
    const float invP = 1.0f / (float)p.P;
    float acc_ce = 0.f, acc_u = 0.f;
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
    for (long long i = 0; i < my_tiles; ++i) {
      const long long tile = blockIdx.x + i * gridDim.x;
      const uint32_t par = (uint32_t)(i & 1);
      const long long prow = tile * kRows + row;
      const bool valid = prow < p.P;
      const float u = nu;
      const int m = nm;
      uint32_t m0[2] = {0, 0}, m1[4] = {0, 0, 0, 0};      // ReLU masks of this thread's columns
      // ---- R1: layer 0 on the FP32 pipes; this thread's hidden units are [64 hf, 64 hf + 64)
      if (i > 0) { mbar_wait(&bar->tile_done, par ^ 1); mbar_wait(&bar->st_done, par ^ 1); fence_after_sync(); }
      {
        float x[F];
#pragma unroll
        for (int k = 0; k < F; ++k) x[k] = nx[k];
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          float v[32];
#pragma unroll
          for (int k = 0; k < 32; ++k) {
            const int j = 64 * hf + 32 * q + k;
            const float4* wr = reinterpret_cast<const float4*>(W0 + j * F);
            float a = b0[j];
#pragma unroll
            for (int c = 0; c < F / 4; ++c) {
              const float4 w = wr[c];
              a = fmaf(w.x, x[4 * c], a); a = fmaf(w.y, x[4 * c + 1], a); a = fmaf(w.z, x[4 * c + 2], a); a = fmaf(w.w, x[4 * c + 3], a);
            }
            if (a > 0.f) m0[q] |= 1u << k;
            v[k] = fmaxf(a, 0.f);
          }
          store_quarter_row(t_h0 + hf * kUnit, row, q, v);
        }
        if (hf == 0) {
          *reinterpret_cast<uint4*>(t_x + sw128_offset(row, 0)) =
              make_uint4(pack_bf16(x[0], x[1]), pack_bf16(x[2], x[3]), pack_bf16(x[4], x[5]), pack_bf16(x[6], x[7]));
          if constexpr (F == 16)
            *reinterpret_cast<uint4*>(t_x + sw128_offset(row, 1)) =
                make_uint4(pack_bf16(x[8], x[9]), pack_bf16(x[10], x[11]), pack_bf16(x[12], x[13]), pack_bf16(x[14], x[15]));
        }
      }
      fence_proxy_async_smem();
      mbar_arrive(&bar->a0_ready);
      if (i + 1 < my_tiles) fetch(tile + gridDim.x);
      // ---- R2: h1 = relu(pre1 + b1): columns [64 hf, +64) from S0, 128 + [32 hf, +32) from S1, 192 + [32 hf, +32) from S0
      mbar_wait(&bar->s0_full, 0);
      fence_after_sync();
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        uint32_t r[32];
        tmem_ld32(lane_addr + kCS0 + 64 * hf + 32 * q, r);
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) {
          const float a = __uint_as_float(r[k]) + b1[64 * hf + 32 * q + k];
          if (a > 0.f) m1[q] |= 1u << k;
          v[k] = fmaxf(a, 0.f);
        }
        store_quarter_row(t_h1 + hf * kUnit, row, q, v);
      }
      fence_before_sync();
      mbar_arrive(&bar->s0_free);
      mbar_wait(&bar->s1_full, 0);
      fence_after_sync();
      {
        uint32_t r[32];
        tmem_ld32(lane_addr + kCS1 + 32 * hf, r);
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) {
          const float a = __uint_as_float(r[k]) + b1[128 + 32 * hf + k];
          if (a > 0.f) m1[2] |= 1u << k;
          v[k] = fmaxf(a, 0.f);
        }
        store_quarter_row(t_h1 + 2 * kUnit, row, hf, v);
      }
      mbar_wait(&bar->s0_full, 1);
      fence_after_sync();
      {
        uint32_t r[32];
        tmem_ld32(lane_addr + kCS0 + 32 * hf, r);
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) {
          const float a = __uint_as_float(r[k]) + b1[192 + 32 * hf + k];
          if (a > 0.f) m1[3] |= 1u << k;
          v[k] = fmaxf(a, 0.f);
        }
        store_quarter_row(t_h1 + 3 * kUnit, row, hf, v);
      }
      fence_before_sync();
      fence_proxy_async_smem();
      mbar_arrive(&bar->a1_ready);
      // ---- R3: softmax, cross entropy, dz (as in loss.cu)
      mbar_wait(&bar->s0_full, 0);
      fence_after_sync();
      {
        const int ng = K / 32;
        float z[2][32];
        float mx = -3.0e38f, zm = 0.f;
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          const int g = hf + 2 * t;
          if (g < ng) {
            uint32_t r[32];
            tmem_ld32(lane_addr + kCS0 + g * 32, r);
            tmem_ld_wait();
#pragma unroll
            for (int e = 0; e < 32; ++e) {
              z[t][e] = __uint_as_float(r[e]) + b2[g * 32 + e];
              mx = fmaxf(mx, z[t][e]);
              if (g * 32 + e == m) zm = z[t][e];
            }
          }
        }
        fence_before_sync();
        x_max[hf * kRows + row] = mx;
        x_zm[hf * kRows + row] = zm;
        asm volatile("bar.sync 1, %0;" ::"n"(kNR) : "memory");
        mx = fmaxf(mx, x_max[(hf ^ 1) * kRows + row]);
        zm += x_zm[(hf ^ 1) * kRows + row];
        float sum = 0.f;
#pragma unroll
        for (int t = 0; t < 2; ++t)
          if (hf + 2 * t < ng) {
#pragma unroll
            for (int e = 0; e < 32; ++e) { z[t][e] = __expf(z[t][e] - mx); sum += z[t][e]; }
          }
        x_sum[hf * kRows + row] = sum;
        asm volatile("bar.sync 1, %0;" ::"n"(kNR) : "memory");
        sum += x_sum[(hf ^ 1) * kRows + row];
        const float ce = (mx + __logf(sum)) - zm;
        const float coef = valid ? p.lambda_ce * (1.0f - u) * invP : 0.f;
        const float scale = coef / sum;
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          const int g = hf + 2 * t;
          if (g < ng) {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              float d[8];
#pragma unroll
              for (int e = 0; e < 8; ++e) d[e] = z[t][c * 8 + e] * scale - ((g * 32 + c * 8 + e == m) ? coef : 0.f);
              const int chunk = g * 4 + c;
              *reinterpret_cast<uint4*>(t_dz + (chunk >> 3) * kUnit + sw128_offset(row, chunk & 7)) =
                  make_uint4(pack_bf16(d[0], d[1]), pack_bf16(d[2], d[3]), pack_bf16(d[4], d[5]), pack_bf16(d[6], d[7]));
            }
          }
        }
        if (hf == 0 && valid) {
          acc_ce += ce * (1.0f - u);
          acc_u += u;
          p.dL[prow * CH + 4 + F] = (p.lambda_u - p.lambda_ce * ce) * invP;
        }
      }
      fence_proxy_async_smem();
      mbar_arrive(&bar->dz_ready);
      // ---- R4: dpre1 = dh1 [pre1 > 0] -> into the h1 tile, once dW2's MMAs have read it
      mbar_wait(&bar->s0_full, 1);
      mbar_wait(&bar->w2_done, par);
      fence_after_sync();
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        uint32_t r[32];
        tmem_ld32(lane_addr + kCS0 + 64 * hf + 32 * q, r);
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) v[k] = ((m1[q] >> k) & 1u) ? __uint_as_float(r[k]) : 0.f;
        store_quarter_row(t_h1 + hf * kUnit, row, q, v);
      }
      fence_before_sync();
      mbar_arrive(&bar->s0_free);
      mbar_wait(&bar->s1_full, 1);
      fence_after_sync();
      {
        uint32_t r[32];
        tmem_ld32(lane_addr + kCS1 + 32 * hf, r);
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) v[k] = ((m1[2] >> k) & 1u) ? __uint_as_float(r[k]) : 0.f;
        store_quarter_row(t_h1 + 2 * kUnit, row, hf, v);
      }
      mbar_wait(&bar->s0_full, 0);
      fence_after_sync();
      {
        uint32_t r[32];
        tmem_ld32(lane_addr + kCS0 + 32 * hf, r);
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) v[k] = ((m1[3] >> k) & 1u) ? __uint_as_float(r[k]) : 0.f;
        store_quarter_row(t_h1 + 3 * kUnit, row, hf, v);
      }
      fence_before_sync();
      fence_proxy_async_smem();
      mbar_arrive(&bar->dp1_ready);
      // ---- R5: dpre0 = dh0 [pre0 > 0] -> into the dz tile; dx = W0^T dpre0
      mbar_wait(&bar->s0_full, 1);
      fence_after_sync();
      float dx[F];
#pragma unroll
      for (int k = 0; k < F; ++k) dx[k] = 0.f;
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        uint32_t r[32];
        tmem_ld32(lane_addr + kCS0 + 64 * hf + 32 * q, r);
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) {
          v[k] = ((m0[q] >> k) & 1u) ? __uint_as_float(r[k]) : 0.f;
          const float4* wr = reinterpret_cast<const float4*>(W0 + (64 * hf + 32 * q + k) * F);
#pragma unroll
          for (int c = 0; c < F / 4; ++c) {
            const float4 w = wr[c];
            dx[4 * c] = fmaf(w.x, v[k], dx[4 * c]); dx[4 * c + 1] = fmaf(w.y, v[k], dx[4 * c + 1]);
            dx[4 * c + 2] = fmaf(w.z, v[k], dx[4 * c + 2]); dx[4 * c + 3] = fmaf(w.w, v[k], dx[4 * c + 3]);
          }
        }
        store_quarter_row(t_dz + hf * kUnit, row, q, v);
      }
      fence_before_sync();
      fence_proxy_async_smem();
      mbar_arrive(&bar->dp0_ready);
      if (hf == 1) {
#pragma unroll
        for (int k = 0; k < F; ++k) *dx_slot(t_x, row, k) = dx[k];
      }
      asm volatile("bar.sync 1, %0;" ::"n"(kNR) : "memory");
      if (hf == 0 && valid) {
        float* o = p.dL + prow * CH + 4;
#pragma unroll
        for (int k = 0; k < F; k += 4)
          *reinterpret_cast<float4*>(o + k) = make_float4(dx[k] + *dx_slot(t_x, row, k), dx[k + 1] + *dx_slot(t_x, row, k + 1),
                                                          dx[k + 2] + *dx_slot(t_x, row, k + 2), dx[k + 3] + *dx_slot(t_x, row, k + 3));
      }
    }
    // ---- end of the CTA's tiles: weight gradients leave TMEM, losses are reduced
    mbar_wait(&bar->tile_done, (uint32_t)((my_tiles - 1) & 1));
    fence_after_sync();
    {
      uint32_t r[32];
      // dW2 [K][256]: lane = code; this thread takes hidden1 [128 hf, 128 hf + 128)
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        tmem_ld32(lane_addr + kCDW2 + 128 * hf + 32 * q, r);
        tmem_ld_wait();
        if (row < K) {
#pragma unroll
          for (int e = 0; e < 32; ++e) atomicAdd(p.dw2 + (size_t)row * kH1 + 128 * hf + 32 * q + e, __uint_as_float(r[e]));
        }
      }
      if (hf == 0) {
        tmem_ld32(lane_addr + kCDb2, r);      // column F of dz^T [x | 1]
        tmem_ld_wait();
        if (row < K && p.db2) atomicAdd(p.db2 + row, __uint_as_float(r[F]));
      } else {
        tmem_ld32(lane_addr + kCDW0, r);      // lane = hidden0 unit: columns 0..F-1 = dW0, column F = db0
        tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < F; ++e) atomicAdd(p.dw0 + (size_t)row * F + e, __uint_as_float(r[e]));
        if (p.db0) atomicAdd(p.db0 + row, __uint_as_float(r[F]));
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
  if (warp == 0) { fence_after_sync(); tmem_dealloc(tmem, 512); }
}

// ------------------------------------------------------------------------------------------------------------------
// dW1 += dpre1^T h0, db1 += dpre1^T 1 from the saved tiles
struct Dw1Barriers {
  uint64_t full[2], empty[2], done;
  uint32_t tmem_base;
};
constexpr int kDw1Stage = 6 * kUnit;
constexpr int kDw1Ones = 2 * kDw1Stage;
constexpr int kDw1Bars = kDw1Ones + kUnit;
constexpr int kDw1Smem = kDw1Bars + 128;
constexpr int kDw1Threads = 32 * 6;

__global__ void __launch_bounds__(kDw1Threads, 1) loss3_dw1_kernel(const uint8_t* __restrict__ save, long long num_tiles,
                                                                    float* __restrict__ dw1, float* __restrict__ db1) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  Dw1Barriers* bar = reinterpret_cast<Dw1Barriers*>(smem + kDw1Bars);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long my_tiles = (num_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x;
  if (threadIdx.x == 0) {
    mbar_init(&bar->full[0], 1); mbar_init(&bar->full[1], 1); mbar_init(&bar->empty[0], 1); mbar_init(&bar->empty[1], 1);
    mbar_init(&bar->done, 1);
    fence_barrier_init();
  }
  if (warp == 1) { tmem_alloc(&bar->tmem_base, 512); tmem_relinquish(); }
  // the ones tile: column 0 of every row = 1.0 (bf16), everything else zero
  for (int i = threadIdx.x; i < kUnit / 16; i += kDw1Threads) reinterpret_cast<uint4*>(smem + kDw1Ones)[i] = make_uint4(0, 0, 0, 0);
  __syncthreads();
  if (threadIdx.x < kRows) *reinterpret_cast<uint16_t*>(smem + kDw1Ones + sw128_offset(threadIdx.x, 0)) = 0x3f80;
  fence_proxy_async_smem();
  fence_before_sync();
  __syncthreads();
  fence_after_sync();
  const uint32_t tmem = bar->tmem_base;
  if (warp == 0) {
    for (long long i = 0; i < my_tiles; ++i) {
      const int s = (int)(i & 1);
      mbar_wait(&bar->empty[s], (uint32_t)(((i >> 1) & 1) ^ 1));
      if (lane == 0) {
        const uint8_t* src = save + (size_t)(blockIdx.x + i * gridDim.x) * kSaveTile;
        mbar_arrive_expect_tx(&bar->full[s], kDw1Stage);
        for (int j = 0; j < 6; ++j) bulk_g2s(smem + s * kDw1Stage + j * kUnit, src + (size_t)j * kUnit, kUnit, &bar->full[s]);
      }
      __syncwarp();
    }
  } else if (warp == 1) {
    const uint32_t hiMN = desc_hi_sw128(1024);
    const uint32_t base = smem_u32(smem);
    const uint32_t onesT = desc_lo(base + kDw1Ones, kUnit);
    const uint32_t id_dw = make_idesc_bf16_major(128, 128, 1, 1), id_side = make_idesc_bf16_major(128, 32, 1, 1);
    auto gemm_rows = [&](uint32_t dcol, uint32_t aT, uint32_t bT, uint32_t idesc, uint32_t acc) {
      for (int k = 0; k < kRows / 16; ++k) {
        const uint32_t off = (uint32_t)k * (2048u >> 4);
        umma_bf16_desc(tmem + dcol, aT + off, hiMN, bT + off, hiMN, idesc, acc | (k ? 1u : 0u));
      }
    };
    for (long long i = 0; i < my_tiles; ++i) {
      const int s = (int)(i & 1);
      mbar_wait(&bar->full[s], (uint32_t)((i >> 1) & 1));
      fence_after_sync();
      if (lane == 0) {
        const uint32_t st = base + s * kDw1Stage, acc = i > 0 ? 1u : 0u;
        const uint32_t h0T = desc_lo(st, kUnit), dpT0 = desc_lo(st + 2 * kUnit, kUnit), dpT1 = desc_lo(st + 4 * kUnit, kUnit);
        gemm_rows(0, dpT0, h0T, id_dw, acc);        // dW1[0:128, :]
        gemm_rows(128, dpT1, h0T, id_dw, acc);      // dW1[128:256, :]
        gemm_rows(256, dpT0, onesT, id_side, acc);  // db1[0:128] in column 0
        gemm_rows(288, dpT1, onesT, id_side, acc);
        umma_commit(&bar->empty[s]);
      }
      __syncwarp();
    }
    if (lane == 0) umma_commit(&bar->done);
    __syncwarp();
  } else {
    const int row = 32 * (warp & 3) + lane;
    const uint32_t lane_addr = tmem + ((uint32_t)(32 * (warp & 3)) << 16);
    mbar_wait(&bar->done, 0);
    fence_after_sync();
    uint32_t r[32];
#pragma unroll
    for (int hv = 0; hv < 2; ++hv) {
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        tmem_ld32(lane_addr + 128 * hv + 32 * q, r);
        tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < 32; ++e) atomicAdd(dw1 + (size_t)(128 * hv + row) * kH0 + 32 * q + e, __uint_as_float(r[e]));
      }
      tmem_ld32(lane_addr + 256 + 32 * hv, r);
      tmem_ld_wait();
      if (db1) atomicAdd(db1 + 128 * hv + row, __uint_as_float(r[0]));
    }
    fence_before_sync();
  }
  __syncthreads();
  if (warp == 1) { fence_after_sync(); tmem_dealloc(tmem, 512); }
}

}  // namespace

size_t legs_loss3_workspace_bytes(int64_t P) {
  const size_t tiles = (size_t)((P + kRows - 1) / kRows);
  return kWsSave + tiles * kSaveTile;
}

int legs_loss3_check(const legs_decoder* dec, int sem_dim) {
  if ((sem_dim != 8 && sem_dim != 16) || dec->in_dim != sem_dim) return LEGS_ERR_DIM;
  if (dec->hidden[0] != kH0 || dec->hidden[1] != kH1) return LEGS_ERR_DIM;
  if (dec->n_codes != 32 && dec->n_codes != 64 && dec->n_codes != 128) return LEGS_ERR_DIM;
  return LEGS_OK;
}

int legs_loss3_launch(legs_ctx* ctx, const float* pixels, int64_t P, int32_t sem_dim, const int32_t* index_map,
                      const legs_decoder* dec, float lambda_ce, float lambda_u, float* dL_dpixels, const legs_decoder_grads* grads,
                      float* loss, void* workspace, cudaStream_t st) {
  uint8_t* ws = (uint8_t*)workspace;
  float* consts = (float*)(ws + kWsConsts);
  loss3_pack_kernel<<<32, 256, 0, st>>>(dec->w[0], dec->b[0], dec->w[1], dec->b[1], dec->w[2], dec->b[2], sem_dim, dec->n_codes, ws,
                                        consts);
  LEGS_LAUNCH_CHECK(ctx);
  Loss3Params lp;
  lp.P = P; lp.num_tiles = (P + kRows - 1) / kRows;
  lp.F = sem_dim; lp.CH = legs_pixel_channels(sem_dim); lp.K = dec->n_codes;
  lp.pixels = pixels; lp.index = index_map; lp.wpack = ws; lp.consts = consts; lp.save = ws + kWsSave;
  lp.lambda_ce = lambda_ce; lp.lambda_u = lambda_u; lp.dL = dL_dpixels;
  lp.dw0 = grads->dw[0]; lp.db0 = grads->db[0]; lp.dw1 = grads->dw[1]; lp.db1 = grads->db[1];
  lp.dw2 = grads->dw[2]; lp.db2 = grads->db[2];
  lp.loss = loss;
  const int smem_bytes = kLoss3Smem + 1024;
  const int grid = (int)(lp.num_tiles < ctx->num_sms ? lp.num_tiles : ctx->num_sms);
  if (sem_dim == 8) {
    LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(loss3_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
    loss3_kernel<8><<<grid, kThreads, smem_bytes, st>>>(lp);
  } else {
    LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(loss3_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
    loss3_kernel<16><<<grid, kThreads, smem_bytes, st>>>(lp);
  }
  LEGS_LAUNCH_CHECK(ctx);
  const int smem_b = kDw1Smem + 1024;
  LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(loss3_dw1_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_b));
  loss3_dw1_kernel<<<grid, kDw1Threads, smem_b, st>>>(lp.save, lp.num_tiles, lp.dw1, lp.db1);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

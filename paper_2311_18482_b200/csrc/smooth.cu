// smooth.cu — adaptive spatial smoothing (SURVEY.md 8(f) item 3; PAPER.md:149-157 Eq. 13-14, :362-370 Table 4), forward and
// reverse mode in one persistent tcgen05 kernel over the Gaussians:
//   h1 = relu(W1 p + b1)                    (fp32 pipes: the input is the 3 coordinates, PE frequency 0)
//   h2 = relu(W2 h1 + b2), h3 = relu(W3 h2 + b3)      (UMMA, A = activation tile K-major, B = weights K-major)
//   s_MLP = W4 h3 + b4                      (fp32 pipes: 8 or 16 outputs)
//   e = s_MLP - s, rho = |e|_2;  L_smo += (1 + max(u, w_s)) rho / n;  g = dL/ds_MLP = lambda e / (n rho);
//   dL/ds = -lambda max(u, w_s) e / (n rho)                                              (Eq. 14, reading C-25)
//   dh3 = W4^T g (fp32 pipes);  dz3 = dh3 [z3 > 0];  dh2 = dz3 W3 (UMMA, B = the SAME W3 tile read MN-major);  dz2; dh1; dz1
//   dW3 += dz3^T h2, dW2 += dz2^T h1 (UMMA over MN-major views: contraction over the tile's 128 Gaussians, accumulated
//   in TMEM over all tiles of the CTA);  dW4^T | . += h3^T [g | p | 1],  . | db3 += dz3^T [g | p | 1],
//   . | db2 += dz2^T [g | p | 1],  . | dW1 | db1 += dz1^T [g | p | 1]   (one shared [128 x 64] side tile U = [g | p | 1]).
// One CTA per SM, 128-Gaussian tiles; warp 0 issues the MMAs, warps 1-8 are 256 row threads (two per Gaussian, 64 hidden
// columns each). All 512 TMEM columns are in use: 128 scratch (z / dh), 128 dW3, 128 dW2, 4 x 32 side accumulators.
#include "common.cuh"
#include "tc05.cuh"

namespace {

using namespace tc05;

constexpr int kRows = 128;
constexpr int kHid = 128;
constexpr int kUnit = 16384;            // [128 rows][64 bf16], 128-byte swizzle
constexpr int kRowWarps = 8;
constexpr int kSmThreads = 32 * (1 + kRowWarps);
// shared-memory units (two per 128-wide activation tile)
constexpr int kUH1 = 0, kUH2 = 2, kUH3 = 4, kUD = 6, kUW2 = 8, kUW3 = 10, kUU = 12, kUnits = 13;
// TMEM columns
constexpr int kCAcc = 0, kCDW3 = 128, kCDW2 = 256, kCS4 = 384, kCS3 = 416, kCS2 = 448, kCS1 = 480;

struct SmoothParams {
  long long n, num_tiles;
  int F;
  const float* means;    // [n,3]
  const float* sem;      // [n,F]
  const float* unc;      // [n]
  const uint8_t* units;  // packed W2, W3 (4 units)
  const float* consts;   // W1 [128][3], b1 [128], b2 [128], b3 [128], W4 [F][128], b4 [F]
  float w_s, lambda;
  float* dsem;           // [n,F]
  int accumulate;        // add into dsem instead of overwriting
  float *dw1, *db1, *dw2, *db2, *dw3, *db3, *dw4, *db4;
  float* loss;
};

__device__ __forceinline__ float bf16f(uint16_t v) { return __uint_as_float((uint32_t)v << 16); }

// weights -> B units (W2, W3: [n = out][k = in], K-major) + fp32 constants
__global__ void __launch_bounds__(256) smooth_pack_kernel(const uint16_t* __restrict__ w1, const float* __restrict__ b1,
                                                          const uint16_t* __restrict__ w2, const float* __restrict__ b2,
                                                          const uint16_t* __restrict__ w3, const float* __restrict__ b3,
                                                          const uint16_t* __restrict__ w4, const float* __restrict__ b4, int F,
                                                          uint8_t* units, float* consts) {
  const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
  for (int c = tid; c < 4 * (kUnit / 16); c += nth) {
    const int u = c / (kUnit / 16), w = c % (kUnit / 16);
    const int r = w / 8, ch = w % 8;
    const uint16_t* src = (u < 2 ? w2 : w3) + (size_t)r * kHid + (u & 1) * 64 + ch * 8;
    *reinterpret_cast<uint4*>(units + (size_t)u * kUnit + sw128_offset((uint32_t)r, (uint32_t)ch)) = *reinterpret_cast<const uint4*>(src);
  }
  float* c1 = consts;                    // W1 [128][3]
  float* cb1 = c1 + kHid * 3;
  float* cb2 = cb1 + kHid;
  float* cb3 = cb2 + kHid;
  float* c4 = cb3 + kHid;                // W4 [F][128]
  float* cb4 = c4 + F * kHid;
  for (int i = tid; i < kHid * 3; i += nth) c1[i] = bf16f(w1[i]);
  for (int i = tid; i < kHid; i += nth) { cb1[i] = b1 ? b1[i] : 0.f; cb2[i] = b2 ? b2[i] : 0.f; cb3[i] = b3 ? b3[i] : 0.f; }
  for (int i = tid; i < F * kHid; i += nth) c4[i] = bf16f(w4[i]);
  for (int i = tid; i < F; i += nth) cb4[i] = b4 ? b4[i] : 0.f;
}

struct SmoothBarriers {
  uint64_t a1_ready, a2_ready, z_ready, b3_ready, b2_ready, b1_ready, g_ready, tile_done;
  uint32_t tmem_base;
};

constexpr int kOffConsts = kUnits * kUnit;                                  // fp32 constants: 384 + 384 + 16*128 + 16 floats max
constexpr int kConstFloats = kHid * 3 + 3 * kHid + 16 * kHid + 16;
constexpr int kOffBars = kOffConsts + ((kConstFloats * 4 + 15) / 16) * 16;
constexpr int kSmoothSmem = kOffBars + 128;

// The pair exchange of s_MLP (16 floats per row) lives in the logical 16-byte chunks 4..7 of the side tile's rows: the
// side MMAs read N = 32 columns = chunks 0..3 only, and the swizzle keeps the chunks of a row apart.
__device__ __forceinline__ float* xch_slot(uint8_t* t_u, int row, int f) {
  return reinterpret_cast<float*>(t_u + sw128_offset((uint32_t)row, (uint32_t)(4 + (f >> 2)))) + (f & 3);
}

// 32 fp32 values (columns 64 hf + 32 q + [0, 32) of the row) -> bf16 -> four 16-byte chunks of the row in a two-unit
// [128 x 128] K-major tile
__device__ __forceinline__ void store_quarter_row(uint8_t* tile, int row, int hf, int q, const float (&v)[32]) {
  uint8_t* unit = tile + hf * kUnit;
#pragma unroll
  for (int c = 0; c < 4; ++c)
    *reinterpret_cast<uint4*>(unit + sw128_offset(row, 4 * q + c)) =
        make_uint4(pack_bf16(v[8 * c], v[8 * c + 1]), pack_bf16(v[8 * c + 2], v[8 * c + 3]), pack_bf16(v[8 * c + 4], v[8 * c + 5]),
                   pack_bf16(v[8 * c + 6], v[8 * c + 7]));
}

template <int F>
__global__ void __launch_bounds__(kSmThreads, 1) smooth_kernel(const __grid_constant__ SmoothParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  float* s_consts = reinterpret_cast<float*>(smem + kOffConsts);
  SmoothBarriers* bar = reinterpret_cast<SmoothBarriers*>(smem + kOffBars);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long my_tiles = (p.num_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x;
  constexpr int NS = F + 4;            // side tile columns in use: g [F], p [3], 1
  constexpr int NSP = 32;              // side accumulator width (columns of one N = 32 MMA)

  if (threadIdx.x == 0) {
    mbar_init(&bar->a1_ready, kRowWarps * 32); mbar_init(&bar->a2_ready, kRowWarps * 32); mbar_init(&bar->z_ready, 1);
    mbar_init(&bar->b3_ready, kRowWarps * 32); mbar_init(&bar->b2_ready, kRowWarps * 32); mbar_init(&bar->b1_ready, kRowWarps * 32);
    mbar_init(&bar->g_ready, 1); mbar_init(&bar->tile_done, 1);
    fence_barrier_init();
  }
  if (warp == 0) { tmem_alloc(&bar->tmem_base, 512); tmem_relinquish(); }
  // zero the activation / side tiles (padding columns of U stay zero for the whole kernel), load the weights and constants
  for (int i = threadIdx.x; i < kUW2 * (kUnit / 16); i += kSmThreads) reinterpret_cast<uint4*>(smem)[i] = make_uint4(0, 0, 0, 0);
  for (int i = threadIdx.x; i < kUnit / 16; i += kSmThreads) reinterpret_cast<uint4*>(smem + kUU * kUnit)[i] = make_uint4(0, 0, 0, 0);
  for (int i = threadIdx.x; i < 4 * (kUnit / 16); i += kSmThreads)
    reinterpret_cast<uint4*>(smem + kUW2 * kUnit)[i] = reinterpret_cast<const uint4*>(p.units)[i];
  for (int i = threadIdx.x; i < kHid * 3 + 3 * kHid + F * kHid + F; i += kSmThreads) s_consts[i] = p.consts[i];
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
    constexpr uint32_t kUnitLo = kUnit >> 4;
    // K-major views (one descriptor per 64-wide k-block unit)
    const uint32_t h1_lo = desc_lo(base + kUH1 * kUnit, 16), h2_lo = desc_lo(base + kUH2 * kUnit, 16);
    const uint32_t h3_lo = desc_lo(base + kUH3 * kUnit, 16), d_lo = desc_lo(base + kUD * kUnit, 16);
    const uint32_t w2_lo = desc_lo(base + kUW2 * kUnit, 16), w3_lo = desc_lo(base + kUW3 * kUnit, 16);
    // MN-major views: LBO = 16 KB between the two 64-wide M/N groups of a tile
    const uint32_t h1T = desc_lo(base + kUH1 * kUnit, kUnit), h2T = desc_lo(base + kUH2 * kUnit, kUnit);
    const uint32_t h3T = desc_lo(base + kUH3 * kUnit, kUnit), dT = desc_lo(base + kUD * kUnit, kUnit);
    const uint32_t w2T = desc_lo(base + kUW2 * kUnit, kUnit), w3T = desc_lo(base + kUW3 * kUnit, kUnit);
    const uint32_t uT = desc_lo(base + kUU * kUnit, kUnit);
    const uint32_t id_fwd = make_idesc_bf16(kRows, kHid);                       // A K-major, B K-major
    const uint32_t id_dx = make_idesc_bf16_major(kRows, kHid, 0, 1);            // A K-major (dz), B MN-major (W read transposed)
    const uint32_t id_dw = make_idesc_bf16_major(kHid, kHid, 1, 1);             // both MN-major: contraction over the rows
    const uint32_t id_side = make_idesc_bf16_major(kHid, NSP, 1, 1);
    uint32_t par = 0;
    auto kmajor_gemm = [&](uint32_t dcol, uint32_t a_lo, uint32_t b_lo, uint32_t idesc, bool b_mn) {
      // contraction over 128 = 8 K steps of 16; K-major operand: 4 steps per unit (+32 B each), then the next unit;
      // MN-major B (W transposed): 16 K rows = +2048 B per step
      for (int k = 0; k < 8; ++k) {
        const uint32_t ao = (k >> 2) * kUnitLo + 2 * (k & 3);
        const uint32_t bo = b_mn ? (uint32_t)k * (2048u >> 4) : ao;
        umma_bf16_desc(tmem + dcol, a_lo + ao, hiK, b_lo + bo, b_mn ? hiMN : hiK, idesc, k ? 1u : 0u);
      }
    };
    auto rows_gemm = [&](uint32_t dcol, uint32_t aT, uint32_t bT, uint32_t idesc, uint32_t acc) {
      // contraction over the tile's 128 rows: both operands MN-major, 16 rows = +2048 B per step
      for (int k = 0; k < kRows / 16; ++k) {
        const uint32_t off = (uint32_t)k * (2048u >> 4);
        umma_bf16_desc(tmem + dcol, aT + off, hiMN, bT + off, hiMN, idesc, acc | (k ? 1u : 0u));
      }
    };
    for (long long i = 0; i < my_tiles; ++i, par ^= 1) {
      const uint32_t acc = i > 0 ? 1u : 0u;
      mbar_wait(&bar->a1_ready, par);
      fence_after_sync();
      if (elect_one_sync()) { kmajor_gemm(kCAcc, h1_lo, w2_lo, id_fwd, false); umma_commit(&bar->z_ready); }   // z2 = h1 W2^T
      __syncwarp();
      mbar_wait(&bar->a2_ready, par);
      fence_after_sync();
      if (elect_one_sync()) { kmajor_gemm(kCAcc, h2_lo, w3_lo, id_fwd, false); umma_commit(&bar->z_ready); }   // z3 = h2 W3^T
      __syncwarp();
      mbar_wait(&bar->b3_ready, par);
      fence_after_sync();
      if (elect_one_sync()) {
        rows_gemm(kCS4, h3T, uT, id_side, acc);                   // dW4^T | . += h3^T [g | p | 1]
        kmajor_gemm(kCAcc, d_lo, w3T, id_dx, true);               // dh2 = dz3 W3
        umma_commit(&bar->g_ready);
        rows_gemm(kCDW3, dT, h2T, id_dw, acc);                    // dW3 += dz3^T h2
        rows_gemm(kCS3, dT, uT, id_side, acc);                    // . | db3 += dz3^T [g | p | 1]
      }
      __syncwarp();
      mbar_wait(&bar->b2_ready, par);
      fence_after_sync();
      if (elect_one_sync()) {
        kmajor_gemm(kCAcc, h3_lo, w2T, id_dx, true);              // dh1 = dz2 W2   (dz2 sits in the h3 tile)
        umma_commit(&bar->g_ready);
        rows_gemm(kCDW2, h3T, h1T, id_dw, acc);                   // dW2 += dz2^T h1
        rows_gemm(kCS2, h3T, uT, id_side, acc);                   // . | db2 += dz2^T [g | p | 1]
      }
      __syncwarp();
      mbar_wait(&bar->b1_ready, par);
      fence_after_sync();
      if (elect_one_sync()) {
        rows_gemm(kCS1, dT, uT, id_side, acc);                    // . | dW1 | db1 += dz1^T [g | p | 1]   (dz1 sits in the D tile)
        umma_commit(&bar->tile_done);
      }
      __syncwarp();
    }
  } else {
    // ===================== 256 row threads: Gaussian = TMEM lane, two threads per row split the hidden columns ===========
    const int row = 32 * (warp & 3) + lane;
    const int hf = (warp - 1) >> 2;
    const uint32_t lane_addr = tmem + ((uint32_t)(32 * (warp & 3)) << 16);
    uint8_t* t_h1 = smem + kUH1 * kUnit;
    uint8_t* t_h2 = smem + kUH2 * kUnit;
    uint8_t* t_h3 = smem + kUH3 * kUnit;
    uint8_t* t_d = smem + kUD * kUnit;
    uint8_t* t_u = smem + kUU * kUnit;
    const float* W1 = s_consts;
    const float* b1 = W1 + kHid * 3;
    const float* b2 = b1 + kHid;
    const float* b3 = b2 + kHid;
    const float* W4 = b3 + kHid;
    const float* b4 = W4 + F * kHid;
    const float invn = 1.0f / (float)p.n;
    float acc_loss = 0.f;
    float acc_db4[F];
#pragma unroll
    for (int f = 0; f < F; ++f) acc_db4[f] = 0.f;
    uint32_t par = 0;
    const int j0 = 64 * hf;            // this thread's hidden columns [j0, j0 + 64)
    for (long long i = 0; i < my_tiles; ++i, par ^= 1) {
      const long long tile = blockIdx.x + i * gridDim.x;
      const long long g = tile * kRows + row;
      const bool valid = g < p.n;
      float px = 0.f, py = 0.f, pz = 0.f, u = 0.f;
      float s[F];
#pragma unroll
      for (int f = 0; f < F; ++f) s[f] = 0.f;
      if (valid) {
        px = p.means[3 * g]; py = p.means[3 * g + 1]; pz = p.means[3 * g + 2];
        u = p.unc[g];
#pragma unroll
        for (int f = 0; f < F; f += 4) {
          const float4 q = *reinterpret_cast<const float4*>(p.sem + g * F + f);
          s[f] = q.x; s[f + 1] = q.y; s[f + 2] = q.z; s[f + 3] = q.w;
        }
      }
      // ---- P1: first layer on the FP32 pipes (32 columns at a time: 2 x 32 of this thread's 64)
      uint32_t m1[2] = {0, 0}, m2[2] = {0, 0}, m3[2] = {0, 0};   // ReLU masks of this thread's 64 columns
      if (i > 0) { mbar_wait(&bar->tile_done, par ^ 1); fence_after_sync(); }   // the last tile's MMAs have read every tile
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        float v[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) {
          const int j = j0 + 32 * q + k;
          const float a = fmaf(W1[3 * j], px, fmaf(W1[3 * j + 1], py, fmaf(W1[3 * j + 2], pz, b1[j])));
          if (a > 0.f) m1[q] |= 1u << k;
          v[k] = fmaxf(a, 0.f);
        }
        store_quarter_row(t_h1, row, hf, q, v);
      }
      if (hf == 0) {   // side tile columns F..F+3 = p, 1 (bf16); a row beyond n contributes nothing: its dz and g are 0
        uint16_t* urow = reinterpret_cast<uint16_t*>(t_u + sw128_offset(row, F >> 3)) + (F & 7);
        const uint32_t a = pack_bf16(px, py), b = pack_bf16(pz, 1.0f);
        urow[0] = (uint16_t)(a & 0xffffu); urow[1] = (uint16_t)(a >> 16); urow[2] = (uint16_t)(b & 0xffffu); urow[3] = (uint16_t)(b >> 16);
      }
      fence_proxy_async_smem();
      mbar_arrive(&bar->a1_ready);
      // ---- P2: h2 = relu(z2 + b2)
      mbar_wait(&bar->z_ready, 0);
      fence_after_sync();
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        uint32_t r[32];
        tmem_ld32(lane_addr + kCAcc + j0 + 32 * q, r);
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) {
          const float a = __uint_as_float(r[k]) + b2[j0 + 32 * q + k];
          if (a > 0.f) m2[q] |= 1u << k;
          v[k] = fmaxf(a, 0.f);
        }
        store_quarter_row(t_h2, row, hf, q, v);
      }
      fence_before_sync();
      fence_proxy_async_smem();
      mbar_arrive(&bar->a2_ready);
      // ---- P3: h3 = relu(z3 + b3), s_MLP = W4 h3 + b4, loss, g, dz3
      mbar_wait(&bar->z_ready, 1);
      fence_after_sync();
      float part[F];
#pragma unroll
      for (int f = 0; f < F; ++f) part[f] = 0.f;
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        uint32_t r[32];
        tmem_ld32(lane_addr + kCAcc + j0 + 32 * q, r);
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) {
          const float a = __uint_as_float(r[k]) + b3[j0 + 32 * q + k];
          if (a > 0.f) m3[q] |= 1u << k;
          v[k] = fmaxf(a, 0.f);
#pragma unroll
          for (int f = 0; f < F; ++f) part[f] = fmaf(W4[f * kHid + j0 + 32 * q + k], v[k], part[f]);
        }
        store_quarter_row(t_h3, row, hf, q, v);
      }
      fence_before_sync();
      // exchange the two halves of s_MLP through shared memory
      if (hf == 1) {
#pragma unroll
        for (int f = 0; f < F; ++f) *xch_slot(t_u, row, f) = part[f];
      }
      asm volatile("bar.sync 1, %0;" ::"n"(kRowWarps * 32) : "memory");
      if (hf == 0) {
#pragma unroll
        for (int f = 0; f < F; ++f) part[f] += *xch_slot(t_u, row, f) + b4[f];
      }
      asm volatile("bar.sync 1, %0;" ::"n"(kRowWarps * 32) : "memory");
      if (hf == 0) {
#pragma unroll
        for (int f = 0; f < F; ++f) *xch_slot(t_u, row, f) = part[f];
      }
      asm volatile("bar.sync 1, %0;" ::"n"(kRowWarps * 32) : "memory");
      float gs[F];   // g = dL/ds_MLP
      {
        float e[F], rho2 = 0.f;
#pragma unroll
        for (int f = 0; f < F; ++f) { e[f] = *xch_slot(t_u, row, f) - s[f]; rho2 = fmaf(e[f], e[f], rho2); }
        const float rho = sqrtf(rho2);
        const float wgt = fmaxf(u, p.w_s);
        const float inv = (valid && rho > 0.f) ? p.lambda * invn / rho : 0.f;
#pragma unroll
        for (int f = 0; f < F; ++f) gs[f] = e[f] * inv;
        if (hf == 0 && valid) {
          acc_loss += (1.0f + wgt) * rho;
          float* o = p.dsem + g * F;
#pragma unroll
          for (int f = 0; f < F; f += 4) {
            float4 q4 = make_float4(-wgt * gs[f], -wgt * gs[f + 1], -wgt * gs[f + 2], -wgt * gs[f + 3]);
            if (p.accumulate) {
              const float4 old = *reinterpret_cast<const float4*>(o + f);
              q4.x += old.x; q4.y += old.y; q4.z += old.z; q4.w += old.w;
            }
            *reinterpret_cast<float4*>(o + f) = q4;
          }
#pragma unroll
          for (int f = 0; f < F; ++f) acc_db4[f] += gs[f];
        }
        if (hf == 0) {   // side tile columns 0..F-1 = g (bf16)
#pragma unroll
          for (int c = 0; c < F / 8; ++c)
            *reinterpret_cast<uint4*>(t_u + sw128_offset(row, c)) =
                make_uint4(pack_bf16(gs[8 * c], gs[8 * c + 1]), pack_bf16(gs[8 * c + 2], gs[8 * c + 3]),
                           pack_bf16(gs[8 * c + 4], gs[8 * c + 5]), pack_bf16(gs[8 * c + 6], gs[8 * c + 7]));
        }
      }
      // dz3 = (W4^T g) [z3 > 0]
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        float v[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) {
          float a = 0.f;
#pragma unroll
          for (int f = 0; f < F; ++f) a = fmaf(W4[f * kHid + j0 + 32 * q + k], gs[f], a);
          v[k] = ((m3[q] >> k) & 1u) ? a : 0.f;
        }
        store_quarter_row(t_d, row, hf, q, v);
      }
      fence_proxy_async_smem();
      mbar_arrive(&bar->b3_ready);
      // ---- P4: dz2 = dh2 [z2 > 0]  -> into the h3 tile (its readers finished before g_ready)
      mbar_wait(&bar->g_ready, 0);
      fence_after_sync();
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        uint32_t r[32];
        tmem_ld32(lane_addr + kCAcc + j0 + 32 * q, r);
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) v[k] = ((m2[q] >> k) & 1u) ? __uint_as_float(r[k]) : 0.f;
        store_quarter_row(t_h3, row, hf, q, v);
      }
      fence_before_sync();
      fence_proxy_async_smem();
      mbar_arrive(&bar->b2_ready);
      // ---- P5: dz1 = dh1 [z1 > 0]  -> into the D tile (dz3's readers finished before the second g_ready)
      mbar_wait(&bar->g_ready, 1);
      fence_after_sync();
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        uint32_t r[32];
        tmem_ld32(lane_addr + kCAcc + j0 + 32 * q, r);
        tmem_ld_wait();
        float v[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) v[k] = ((m1[q] >> k) & 1u) ? __uint_as_float(r[k]) : 0.f;
        store_quarter_row(t_d, row, hf, q, v);
      }
      fence_before_sync();
      fence_proxy_async_smem();
      mbar_arrive(&bar->b1_ready);
    }
    // ---- end of the CTA's tiles: weight gradients leave TMEM (lane = output unit of the layer), loss is reduced
    mbar_wait(&bar->tile_done, par ^ 1);
    fence_after_sync();
    {
      uint32_t r[32];
      // dW3 [o][j], dW2 [o][j]: lane = o, columns = j; this thread takes j in [64 hf, 64 hf + 64)
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        tmem_ld32(lane_addr + kCDW3 + j0 + 32 * q, r);
        tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < 32; ++e) atomicAdd(p.dw3 + (size_t)row * kHid + j0 + 32 * q + e, __uint_as_float(r[e]));
        tmem_ld32(lane_addr + kCDW2 + j0 + 32 * q, r);
        tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < 32; ++e) atomicAdd(p.dw2 + (size_t)row * kHid + j0 + 32 * q + e, __uint_as_float(r[e]));
      }
      if (hf == 0) {
        tmem_ld32(lane_addr + kCS4, r);      // lane = hidden j: columns 0..F-1 = dW4[f][j]
        tmem_ld_wait();
#pragma unroll
        for (int f = 0; f < F; ++f) atomicAdd(p.dw4 + (size_t)f * kHid + row, __uint_as_float(r[f]));
        tmem_ld32(lane_addr + kCS3, r);      // column F+3 = db3[o]
        tmem_ld_wait();
        if (p.db3) atomicAdd(p.db3 + row, __uint_as_float(r[F + 3]));
      } else {
        tmem_ld32(lane_addr + kCS2, r);      // column F+3 = db2[o]
        tmem_ld_wait();
        if (p.db2) atomicAdd(p.db2 + row, __uint_as_float(r[F + 3]));
        tmem_ld32(lane_addr + kCS1, r);      // columns F..F+2 = dW1[j][0..2], column F+3 = db1[j]
        tmem_ld_wait();
#pragma unroll
        for (int k = 0; k < 3; ++k) atomicAdd(p.dw1 + (size_t)row * 3 + k, __uint_as_float(r[F + k]));
        if (p.db1) atomicAdd(p.db1 + row, __uint_as_float(r[F + 3]));
      }
    }
    fence_before_sync();
    for (int o = 16; o > 0; o >>= 1) {
      acc_loss += __shfl_xor_sync(0xffffffffu, acc_loss, o);
#pragma unroll
      for (int f = 0; f < F; ++f) acc_db4[f] += __shfl_xor_sync(0xffffffffu, acc_db4[f], o);
    }
    if (lane == 0 && hf == 0) {
      atomicAdd(p.loss, acc_loss * invn);
      if (p.db4) {
#pragma unroll
        for (int f = 0; f < F; ++f) atomicAdd(p.db4 + f, acc_db4[f]);
      }
    }
  }
  fence_before_sync();
  __syncthreads();
  if (warp == 0) { fence_after_sync(); tmem_dealloc(tmem, 512); }
}

}  // namespace

extern "C" {

size_t legs_smooth_workspace_bytes(int32_t sem_dim) {
  (void)sem_dim;
  return (size_t)4 * kUnit + (size_t)kConstFloats * 4 + 256;
}

int legs_smooth_loss(legs_ctx* ctx, int64_t n, int32_t sem_dim, const float* means, const float* sem, const float* unc,
                     const legs_smooth_mlp* mlp, float w_s, float lambda_smo, int32_t accumulate, float* dsem,
                     const legs_smooth_grads* grads, float* loss, void* workspace, size_t workspace_bytes, void* stream) {
  if (!ctx || !mlp || !grads) return LEGS_ERR_NULL;
  if ((sem_dim != 8 && sem_dim != 16) || mlp->hidden != kHid || n < 0) return LEGS_ERR_DIM;
  if (!means || !sem || !unc || !dsem || !loss || !workspace) return LEGS_ERR_NULL;
  for (int l = 0; l < 4; ++l) {
    if (!mlp->w[l] || !grads->dw[l]) return LEGS_ERR_NULL;
    if (!legs_aligned16(mlp->w[l]) || !legs_aligned16(grads->dw[l]) || (mlp->b[l] && !legs_aligned16(mlp->b[l])) ||
        (grads->db[l] && !legs_aligned16(grads->db[l])))
      return LEGS_ERR_ALIGN;
  }
  if (!legs_aligned16(means) || !legs_aligned16(sem) || !legs_aligned16(unc) || !legs_aligned16(dsem) || !legs_aligned16(loss) ||
      !legs_aligned16(workspace))
    return LEGS_ERR_ALIGN;
  if (workspace_bytes < legs_smooth_workspace_bytes(sem_dim)) return LEGS_ERR_WORKSPACE;
  if (n == 0) return LEGS_OK;
  cudaStream_t st = (cudaStream_t)stream;
  uint8_t* units = (uint8_t*)workspace;
  float* consts = (float*)(units + 4 * kUnit);
  smooth_pack_kernel<<<16, 256, 0, st>>>(mlp->w[0], mlp->b[0], mlp->w[1], mlp->b[1], mlp->w[2], mlp->b[2], mlp->w[3], mlp->b[3],
                                         sem_dim, units, consts);
  LEGS_LAUNCH_CHECK(ctx);
  SmoothParams sp;
  sp.n = n; sp.num_tiles = (n + kRows - 1) / kRows; sp.F = sem_dim;
  sp.means = means; sp.sem = sem; sp.unc = unc; sp.units = units; sp.consts = consts;
  sp.w_s = w_s; sp.lambda = lambda_smo; sp.dsem = dsem; sp.accumulate = accumulate ? 1 : 0;
  sp.dw1 = grads->dw[0]; sp.db1 = grads->db[0]; sp.dw2 = grads->dw[1]; sp.db2 = grads->db[1];
  sp.dw3 = grads->dw[2]; sp.db3 = grads->db[2]; sp.dw4 = grads->dw[3]; sp.db4 = grads->db[3];
  sp.loss = loss;
  const int smem_bytes = kSmoothSmem + 1024;
  const int grid = (int)(sp.num_tiles < ctx->num_sms ? sp.num_tiles : ctx->num_sms);
  if (sem_dim == 8) {
    LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(smooth_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
    smooth_kernel<8><<<grid, kSmThreads, smem_bytes, st>>>(sp);
  } else {
    LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(smooth_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
    smooth_kernel<16><<<grid, kSmThreads, smem_bytes, st>>>(sp);
  }
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

}  // extern "C"

// quantize.cu — quantisation search and codebook losses (SURVEY.md 8(f) item 2; PAPER.md:76-108 Eq. 3-7, :310-329
// Eq. 16-20):
//   D(F, f_i) = cos<F^CLIP, f_i^CLIP> + lambda_DINO cos<F^DINO, f_i^DINO>  (Eq. 4),  m = argmax_i D  (Eq. 16),
//   r = sum onehot(m) / P (Eq. 17),  p = sum softmax(D) / P (Eq. 18-19),  L_lb = sum r o p (Eq. 20),
//   L_cos = mean [(1 - cos_CLIP(m)) + lambda_DINO (1 - cos_DINO(m))] (Eq. 5),  L_q = lambda_cos L_cos + lambda_lb L_lb (Eq. 7).
//
// The search is the dense contraction [P, d] x [d, N] (d = 896, N <= 128): tcgen05.mma with fp32 accumulators in TMEM,
// one accumulator for the CLIP dimensions and one for the DINO dimensions of every tile (the two cosines are scaled by
// different per-pixel norms). HBM-bound: every feature row (2 d bytes) is read once.
//
// One persistent CTA per SM, 128-row tiles. A ring stage holds one 64-wide k-block of the tile's features and of the
// codebook ([128 x 64] bf16 units, 128-byte swizzle, written by TMA tensor loads straight from the caller's arrays; the
// codebook comes from L2). Warp roles: warp 0 TMA producer; warp 1 MMA issuer (+ TMEM); warps 2-9 read each feature unit
// back from shared memory and accumulate the row norms |F^CLIP|^2, |F^DINO|^2 (two threads per row, half a row each);
// warps 10-17 finish the rows: scores, arg max, softmax, per-code probability sums (warp butterfly transpose), histogram.
// The two accumulators of a tile take 256 TMEM columns, so the tiles alternate between two accumulator sets and the
// finishing warps between two groups of four (one per set): the finishing of tile i (two passes over 128 scores per row)
// runs under the loads and MMAs of tiles i + 1 and i + 2, and the HBM stream does not wait for it. (Until round 2's last
// session the kernel worked on pairs of tiles that held all 512 columns: the stream stalled while a pair was finished.)
#include <cuda.h>

#include "common.cuh"
#include "tc05.cuh"
#include "tmap.cuh"

namespace {

using namespace tc05;

constexpr int kRows = 128;
constexpr int kUnitBytes = 16384;        // [128 rows][64 bf16], SW128 K-major
constexpr int kStageBytes = 2 * kUnitBytes;   // features, codebook
constexpr int kStages = 6;
constexpr int kNormWarps = 8, kEpiWarps = 8;
constexpr int kQThreads = 32 * (2 + kNormWarps + kEpiWarps);   // 576
constexpr int kMaxCodes = 128;
constexpr float kLog2e = 1.4426950408889634f;

struct QuantParams {
  long long P, num_tiles;
  int N, d, d_clip;
  float lambda_dino;
  const uint16_t* codebook;
  int32_t* index;
  unsigned int* hist;     // [128]
  float* psum;            // [128]
  float* sums;            // [2]: sum (1 - cos_CLIP(m)), sum (1 - cos_DINO(m))
};

struct QuantBarriers {
  uint64_t full[kStages], empty[kStages];
  uint64_t acc_full[2], acc_empty[2];     // per accumulator set
  uint64_t norm_full[2], norm_empty[2];   // per norm slot (= accumulator set)
  uint32_t tmem_base;
};

__device__ __forceinline__ float ex2_approx(float x) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float bf_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

// 32 values per lane -> lane l keeps the warp total of value l (butterfly transpose reduction, 31 shuffles)
template <int N, int OFF>
__device__ __forceinline__ void col_round(float (&v)[32], int lane) {
  constexpr int H = N / 2;
  const bool upper = (lane & OFF) != 0;
#pragma unroll
  for (int i = 0; i < H; ++i) {
    const float send = upper ? v[i] : v[i + H];
    const float keep = upper ? v[i + H] : v[i];
    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, OFF);
  }
}
__device__ __forceinline__ float column_sums(float (&v)[32], int lane) {
  col_round<32, 16>(v, lane); col_round<16, 8>(v, lane); col_round<8, 4>(v, lane);
  col_round<4, 2>(v, lane);   col_round<2, 1>(v, lane);
  return v[0];
}

__global__ void __launch_bounds__(kQThreads, 1) quantize_kernel(const __grid_constant__ QuantParams p,
                                                                const __grid_constant__ CUtensorMap tmap_feat,
                                                                const __grid_constant__ CUtensorMap tmap_code) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  uint8_t* ring = smem;
  float* s_inv = reinterpret_cast<float*>(ring + kStages * kStageBytes);   // [2][128]: 1/|f_i^CLIP|, 1/|f_i^DINO|
  float* s_norm = s_inv + 2 * kMaxCodes;                                   // [2 slots][2 row halves][128 rows][2]
  unsigned int* s_hist = reinterpret_cast<unsigned int*>(s_norm + 2 * 256 * 2);   // [128]
  float* s_psum = reinterpret_cast<float*>(s_hist + kMaxCodes);            // [128]
  QuantBarriers* bar = reinterpret_cast<QuantBarriers*>(s_psum + kMaxCodes);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int N = p.N, d = p.d, kbs = d / 64, kc = p.d_clip / 64;
  const long long my_tiles = (p.num_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x;

  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) { mbar_init(&bar->full[s], 1); mbar_init(&bar->empty[s], 1 + kNormWarps); }
    for (int b = 0; b < 2; ++b) {
      mbar_init(&bar->acc_full[b], 1); mbar_init(&bar->acc_empty[b], kEpiWarps / 2);
      mbar_init(&bar->norm_full[b], kNormWarps); mbar_init(&bar->norm_empty[b], kEpiWarps / 2);
    }
    fence_barrier_init();
    prefetch_tmap(&tmap_feat);
    prefetch_tmap(&tmap_code);
  }
  if (warp == 1) { tmem_alloc(&bar->tmem_base, 512); tmem_relinquish(); }
  // reciprocal norms of the two parts of every code (fp32 from the bf16 codebook; rows >= N: 0), and zeroed counters
  for (int i = warp; i < kMaxCodes; i += kQThreads / 32) {
    float a = 0.f, b = 0.f;
    if (i < N) {
      const uint16_t* row = p.codebook + (size_t)i * d;
      for (int j = lane; j < d; j += 32) {
        const float x = __uint_as_float((uint32_t)row[j] << 16);
        if (j < p.d_clip) a = fmaf(x, x, a); else b = fmaf(x, x, b);
      }
    }
    for (int o = 16; o > 0; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
    if (lane == 0) { s_inv[i] = i < N ? rsqrtf(fmaxf(a, 1e-30f)) : 0.f; s_inv[kMaxCodes + i] = i < N ? rsqrtf(fmaxf(b, 1e-30f)) : 0.f; }
  }
  for (int i = threadIdx.x; i < kMaxCodes; i += kQThreads) { s_hist[i] = 0u; s_psum[i] = 0.f; }
  fence_before_sync();
  __syncthreads();
  fence_after_sync();
  const uint32_t tmem = bar->tmem_base;

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      int s = 0; uint32_t ph = 0;
      for (long long i = 0; i < my_tiles; ++i) {
        const long long tile = blockIdx.x + i * gridDim.x;
        const int32_t row0 = (int32_t)(tile * kRows);
        for (int kb = 0; kb < kbs; ++kb) {
          mbar_wait(&bar->empty[s], ph ^ 1);
          mbar_arrive_expect_tx(&bar->full[s], (uint32_t)kStageBytes);
          uint8_t* st = ring + s * kStageBytes;
          tma_load_2d(st, &tmap_feat, kb * 64, row0, &bar->full[s]);
          tma_load_2d(st + kUnitBytes, &tmap_code, kb * 64, 0, &bar->full[s]);
          if (++s == kStages) { s = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    int s = 0; uint32_t ph = 0;
    const uint32_t ring_lo = desc_lo_sw128(smem_u32(ring));
    constexpr uint32_t kUnitLo = kUnitBytes >> 4, kStageLo = kStageBytes >> 4;
    const uint32_t idesc = make_idesc_bf16(kRows, (uint32_t)(N < 16 ? 16 : N));
    for (long long i = 0; i < my_tiles; ++i) {
      const uint32_t set = (uint32_t)(i & 1), use = (uint32_t)((i >> 1) & 1);
      mbar_wait(&bar->acc_empty[set], use ^ 1);   // the set's finishing warps have drained the tile before last
      fence_after_sync();
      for (int kb = 0; kb < kbs; ++kb) {
        mbar_wait(&bar->full[s], ph);
        fence_after_sync();
        if (elect_one_sync()) {
          const uint32_t part = set * 256u + (kb < kc ? 0u : 128u);   // CLIP accumulator / DINO accumulator of the set
          const uint32_t first = (kb == 0 || kb == kc) ? 0u : 1u;
          const uint32_t a0 = ring_lo + s * kStageLo, b = a0 + kUnitLo;
#pragma unroll
          for (int k = 0; k < 4; ++k) umma_bf16_lo(tmem + part, a0 + 2 * k, b + 2 * k, idesc, first | (k ? 1u : 0u));
          umma_commit(&bar->empty[s]);
          if (kb == kbs - 1) umma_commit(&bar->acc_full[set]);
        }
        __syncwarp();
        if (++s == kStages) { s = 0; ph ^= 1; }
      }
    }
  } else if (warp < 2 + kNormWarps) {
    // ===================== row norms of the features, from the staged units =====================
    const int t = threadIdx.x - 64;              // 0..255: row t % 128, half of the row's eight 16-byte chunks t / 128
    const int half = t >> 7, row = t & 127;
    const uint32_t row_off = (uint32_t)(row >> 3) * 1024u + (uint32_t)(row & 7) * 128u;
    int s = 0; uint32_t ph = 0;
    for (long long i = 0; i < my_tiles; ++i) {
      float nc = 0.f, nd = 0.f;
      for (int kb = 0; kb < kbs; ++kb) {
        mbar_wait(&bar->full[s], ph);
        const uint8_t* u = ring + s * kStageBytes + row_off;
        float acc0 = 0.f, acc1 = 0.f;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const uint4 q = *reinterpret_cast<const uint4*>(u + (((4 * half + c + row) & 7) << 4));   // rotated: conflict-free
          acc0 = fmaf(bf_lo(q.x), bf_lo(q.x), acc0); acc1 = fmaf(bf_hi(q.x), bf_hi(q.x), acc1);
          acc0 = fmaf(bf_lo(q.y), bf_lo(q.y), acc0); acc1 = fmaf(bf_hi(q.y), bf_hi(q.y), acc1);
          acc0 = fmaf(bf_lo(q.z), bf_lo(q.z), acc0); acc1 = fmaf(bf_hi(q.z), bf_hi(q.z), acc1);
          acc0 = fmaf(bf_lo(q.w), bf_lo(q.w), acc0); acc1 = fmaf(bf_hi(q.w), bf_hi(q.w), acc1);
        }
        if (kb < kc) nc += acc0 + acc1; else nd += acc0 + acc1;
        __syncwarp();
        if (lane == 0) mbar_arrive(&bar->empty[s]);
        if (++s == kStages) { s = 0; ph ^= 1; }
      }
      const int slot = (int)(i & 1);
      mbar_wait(&bar->norm_empty[slot], (uint32_t)(((i >> 1) & 1) ^ 1));
      s_norm[(slot * 256 + t) * 2] = nc;
      s_norm[(slot * 256 + t) * 2 + 1] = nd;
      __syncwarp();
      __threadfence_block();
      if (lane == 0) mbar_arrive(&bar->norm_full[slot]);
    }
  } else {
    // ===================== finishing warps: scores, arg max, softmax, statistics =====================
    const int e = warp - (2 + kNormWarps);       // 0..7
    const int set = e >> 2, row = 32 * (warp & 3) + lane;   // this warp's accumulator set; its quarter of the TMEM lanes
    const uint32_t lane_addr = tmem + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)set * 256u;
    const int ng = N / 32;
    float col_acc[kMaxCodes / 32];
#pragma unroll
    for (int g = 0; g < kMaxCodes / 32; ++g) col_acc[g] = 0.f;
    float sum_c = 0.f, sum_d = 0.f;
    for (long long i = set; i < my_tiles; i += 2) {   // the tiles of this set
      const long long tile = blockIdx.x + i * gridDim.x;
      const long long prow = tile * kRows + row;
      const bool valid = prow < p.P;
      const uint32_t use = (uint32_t)((i >> 1) & 1);
      mbar_wait(&bar->norm_full[set], use);
      const float nc = s_norm[(set * 256 + row) * 2] + s_norm[(set * 256 + 128 + row) * 2];
      const float nd = s_norm[(set * 256 + row) * 2 + 1] + s_norm[(set * 256 + 128 + row) * 2 + 1];
      __syncwarp();
      if (lane == 0) mbar_arrive(&bar->norm_empty[set]);
      const float a = rsqrtf(fmaxf(nc, 1e-30f)), b = rsqrtf(fmaxf(nd, 1e-30f));
      mbar_wait(&bar->acc_full[set], use);
      fence_after_sync();
      // Scores in log2 units, two codes per packed instruction (mul / fma.rn.f32x2: the finishing warps are bound by
      // instruction issue): D log2(e) = (acc_c / |f_c|) (log2(e) / |F_c|) + (acc_d / |f_d|) (lambda log2(e) / |F_d|).
      unsigned long long a2, b2;
      {
        const float al = a * kLog2e, bl = b * (p.lambda_dino * kLog2e);
        asm("mov.b64 %0, {%1, %1};" : "=l"(a2) : "f"(al));
        asm("mov.b64 %0, {%1, %1};" : "=l"(b2) : "f"(bl));
      }
      const uint32_t inv_addr = legs_smem_addr(s_inv);
      // pass 1: arg max (lowest index on ties), partition sum (|D| <= 1 + lambda: no overflow, no max needed)
      float best = -3.0e38f, tcb = 0.f, tdb = 0.f, Z = 0.f;   // best score; acc / |f| of the best code, CLIP and DINO part
      int ibest = 0;
      for (int g = 0; g < ng; ++g) {
        uint32_t rc[32], rd[32];
        tmem_ld32(lane_addr + g * 32, rc);
        tmem_ld32(lane_addr + 128 + g * 32, rd);
        tmem_ld_wait();
#pragma unroll
        for (int k = 0; k < 32; k += 2) {
          const int idx = g * 32 + k;
          unsigned long long vc, vd, t1, t2, sc;
          asm("mov.b64 %0, {%1, %2};" : "=l"(vc) : "r"(rc[k]), "r"(rc[k + 1]));
          asm("mov.b64 %0, {%1, %2};" : "=l"(vd) : "r"(rd[k]), "r"(rd[k + 1]));
          asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(t1) : "l"(vc), "l"(legs_lds64_u64(inv_addr + 4 * idx)));
          asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(t2) : "l"(vd), "l"(legs_lds64_u64(inv_addr + 4 * (kMaxCodes + idx))));
          asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(sc) : "l"(t2), "l"(b2));
          asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(sc) : "l"(t1), "l"(a2));
          float s0, s1, c0, c1, d0, d1;
          asm("mov.b64 {%0, %1}, %2;" : "=f"(s0), "=f"(s1) : "l"(sc));
          asm("mov.b64 {%0, %1}, %2;" : "=f"(c0), "=f"(c1) : "l"(t1));
          asm("mov.b64 {%0, %1}, %2;" : "=f"(d0), "=f"(d1) : "l"(t2));
          if (s0 > best) { best = s0; ibest = idx; tcb = c0; tdb = d0; }
          if (s1 > best) { best = s1; ibest = idx + 1; tcb = c1; tdb = d1; }
          Z += ex2_approx(s0) + ex2_approx(s1);
        }
      }
      const float cbest = tcb * a, dbest = tdb * b;
      // pass 2: probabilities 2^(score - log2 Z) and their per-code sums over the warp's 32 rows
      unsigned long long nlz2;
      {
        const float nlz = valid ? -__log2f(Z) : -200.0f;   // rows beyond P: probability 0
        asm("mov.b64 %0, {%1, %1};" : "=l"(nlz2) : "f"(nlz));
      }
      for (int g = 0; g < ng; ++g) {
        uint32_t rc[32], rd[32];
        tmem_ld32(lane_addr + g * 32, rc);
        tmem_ld32(lane_addr + 128 + g * 32, rd);
        tmem_ld_wait();
        float pr[32];
#pragma unroll
        for (int k = 0; k < 32; k += 2) {
          const int idx = g * 32 + k;
          unsigned long long vc, vd, t1, t2, sc;
          asm("mov.b64 %0, {%1, %2};" : "=l"(vc) : "r"(rc[k]), "r"(rc[k + 1]));
          asm("mov.b64 %0, {%1, %2};" : "=l"(vd) : "r"(rd[k]), "r"(rd[k + 1]));
          asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(t1) : "l"(vc), "l"(legs_lds64_u64(inv_addr + 4 * idx)));
          asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(t2) : "l"(vd), "l"(legs_lds64_u64(inv_addr + 4 * (kMaxCodes + idx))));
          asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(sc) : "l"(t2), "l"(b2), "l"(nlz2));
          asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(sc) : "l"(t1), "l"(a2));
          float s0, s1;
          asm("mov.b64 {%0, %1}, %2;" : "=f"(s0), "=f"(s1) : "l"(sc));
          pr[k] = ex2_approx(s0);
          pr[k + 1] = ex2_approx(s1);
        }
        col_acc[g] += column_sums(pr, lane);
      }
      fence_before_sync();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bar->acc_empty[set]);
      if (valid) {
        p.index[prow] = ibest;
        atomicAdd(&s_hist[ibest], 1u);
        sum_c += 1.0f - cbest;
        sum_d += 1.0f - dbest;
      }
    }
    // the CTA's statistics: shared-memory totals first
#pragma unroll
    for (int g = 0; g < kMaxCodes / 32; ++g)
      if (g < ng && col_acc[g] != 0.f) atomicAdd(&s_psum[g * 32 + lane], col_acc[g]);
    for (int o = 16; o > 0; o >>= 1) { sum_c += __shfl_xor_sync(0xffffffffu, sum_c, o); sum_d += __shfl_xor_sync(0xffffffffu, sum_d, o); }
    if (lane == 0) { atomicAdd(p.sums, sum_c); atomicAdd(p.sums + 1, sum_d); }
  }
  fence_before_sync();
  __syncthreads();
  if (warp == 1) { fence_after_sync(); tmem_dealloc(tmem, 512); }
  for (int i = threadIdx.x; i < N; i += kQThreads) {
    if (s_hist[i]) atomicAdd(p.hist + i, s_hist[i]);
    if (s_psum[i] != 0.f) atomicAdd(p.psum + i, s_psum[i]);
  }
}

// r = hist / P, p = psum / P, L_lb = sum r p, L_cos = (sum_c + lambda_dino sum_d) / P, L_q (one warp)
__global__ void quantize_finish_kernel(const unsigned int* __restrict__ hist, const float* __restrict__ psum,
                                       const float* __restrict__ sums, long long P, int N, float lambda_dino,
                                       float lambda_cos, float lambda_lb, float* r, float* pm, float* loss) {
  const int lane = threadIdx.x;
  const float invP = 1.0f / (float)P;
  float lb = 0.f;
  for (int i = lane; i < N; i += 32) {
    const float ri = (float)hist[i] * invP, pi = psum[i] * invP;
    if (r) r[i] = ri;
    if (pm) pm[i] = pi;
    lb = fmaf(ri, pi, lb);
  }
  for (int o = 16; o > 0; o >>= 1) lb += __shfl_xor_sync(0xffffffffu, lb, o);
  if (lane == 0) {
    const float lcos = (sums[0] + lambda_dino * sums[1]) * invP;
    loss[0] = lcos; loss[1] = lb; loss[2] = lambda_cos * lcos + lambda_lb * lb;
  }
}

}  // namespace

extern "C" {

size_t legs_quantize_workspace_bytes(int32_t N) {
  (void)N;
  return 2 * kMaxCodes * 4 + 256;   // hist [128] u32, psum [128] f32, sums [2] f32
}

int legs_quantize(legs_ctx* ctx, const uint16_t* features, int64_t P, const uint16_t* codebook, int32_t N, int32_t d,
                  int32_t d_clip, float lambda_dino, float lambda_cos, float lambda_lb, int32_t* index_map, float* r,
                  float* p, float* loss, void* workspace, size_t workspace_bytes, void* stream) {
  if (!ctx || !features || !codebook || !index_map || !loss || !workspace) return LEGS_ERR_NULL;
  if (!legs_aligned16(features) || !legs_aligned16(codebook) || !legs_aligned16(index_map) || !legs_aligned16(loss) ||
      !legs_aligned16(workspace) || (r && !legs_aligned16(r)) || (p && !legs_aligned16(p)))
    return LEGS_ERR_ALIGN;
  if ((N != 32 && N != 64 && N != 128) || d < 128 || d > 4096 || (d & 63) || d_clip < 64 || d_clip >= d || (d_clip & 63) || P < 0)
    return LEGS_ERR_DIM;
  if (!(lambda_dino >= 0.f && lambda_dino <= 8.f)) return LEGS_ERR_DIM;   // exp(D) is taken without a max: |D| <= 1 + lambda
  if (workspace_bytes < legs_quantize_workspace_bytes(N)) return LEGS_ERR_WORKSPACE;
  if (P == 0) return LEGS_OK;
  cudaStream_t st = (cudaStream_t)stream;
  LEGS_CUDA_CHECK(ctx, cudaMemsetAsync(workspace, 0, legs_quantize_workspace_bytes(N), st));
  QuantParams qp;
  qp.P = P; qp.num_tiles = (P + kRows - 1) / kRows;
  qp.N = N; qp.d = d; qp.d_clip = d_clip; qp.lambda_dino = lambda_dino;
  qp.codebook = codebook; qp.index = index_map;
  qp.hist = (unsigned int*)workspace;
  qp.psum = (float*)workspace + kMaxCodes;
  qp.sums = (float*)workspace + 2 * kMaxCodes;
  CUtensorMap tf, tc;
  int rc;
  if ((rc = make_tmap_bf16_2d(ctx, features, (uint64_t)d, (uint64_t)P, 64, kRows, &tf)) != LEGS_OK) return rc;
  if ((rc = make_tmap_bf16_2d(ctx, codebook, (uint64_t)d, (uint64_t)N, 64, kRows, &tc)) != LEGS_OK) return rc;
  const int smem_bytes = kStages * kStageBytes + (2 * kMaxCodes + 2 * 256 * 2 + 2 * kMaxCodes) * 4 + 256 + 1024;
  LEGS_CUDA_CHECK(ctx, cudaFuncSetAttribute(quantize_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
  const int grid = (int)(qp.num_tiles < ctx->num_sms ? qp.num_tiles : ctx->num_sms);
  quantize_kernel<<<grid, kQThreads, smem_bytes, st>>>(qp, tf, tc);
  LEGS_LAUNCH_CHECK(ctx);
  quantize_finish_kernel<<<1, 32, 0, st>>>(qp.hist, qp.psum, qp.sums, P, N, lambda_dino, lambda_cos, lambda_lb, r, p, loss);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

}  // extern "C"

// project_backward.cu — S7: per-Gaussian projection + SH backward (BASELINE.json north_star (4) "then the projection
// backward to 3D parameters"). One thread per Gaussian, HBM-streaming.
// Compiled with IEEE division and square root but WITH FMA contraction (build.py: -prec-div -prec-sqrt only), so the
// forward intermediates recomputed here (t, J, Sigma, Sigma') are close to, not bit-identical with, what preprocess.cu
// (compiled without contraction, rule P-0) computed. Nothing here may depend on that: every forward DECISION is taken
// from stored bits - visibility from tiles_touched[], the colour and Jacobian clamps from clamped[] (bits 0-2 / 3-4) - and
// the Cholesky factor R' of the conic comes from the record preprocess.cu wrote. Only smooth quantities are recomputed.
// Do not add a recomputed branch (a clamp test, a cull test) that would have to match the forward pass bit for bit.
#include "common.cuh"

namespace {

constexpr int kBlock = 128;

__device__ __constant__ float kC[10] = {
    0.28209479177387814f, 0.48860251190291992f, 1.0925484305920792f, 0.31539156525252005f, 0.54627421529603959f,
    0.59004358992664352f, 2.8906114426405538f,  0.45704579946446572f, 0.37317633259011540f, 1.4453057213202769f};

struct PbArgs {
  long long n;
  int sh_degree, sh_stored, accumulate, F, RS, RG, geo;
  const float *means, *scales, *quats, *sh;
  const unsigned int* tiles;
  const unsigned char* clamped;
  const float* conic_opacity;
  const float* record;   // [n, RS]: slots 2..4 hold the scaled Cholesky factor R' of the conic (preprocess.cu)
  const float* gscr;     // [n, RG]: S0, Su, Sv, Huu, Huv, Hvv, drgb[3], (ddepth if geo,) dsem[F], dunc reduced by backward.cu
  float *dmeans, *dscales, *dquats, *dsh, *dmean2d, *dopac, *dsem, *dunc;
};

__device__ __forceinline__ void store(float* p, float v, int acc) { *p = acc ? (*p + v) : v; }

__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ bool mbar_done(unsigned long long* bar, unsigned parity) {
  unsigned ok;
  asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(ok) : "r"(smem_addr(bar)), "r"(parity) : "memory");
  return ok != 0;
}

// One Gaussian. `srow` is this Gaussian's SH row in shared memory: coefficients on entry, dL/dSH on exit. BULK: the row
// arrives by a bulk async copy (waited for here, just before the coefficients are read) and is accessed in 16-byte chunks.
template <bool BULK>
__device__ __forceinline__ void project_backward_one(const PbArgs& a, const DevCamera& cam, long long i, float* srow,
                                                     unsigned long long* bar) {
  const int acc = a.accumulate;
  const int nb = (a.sh_degree + 1) * (a.sh_degree + 1);
  const float* W = cam.W;
  const float px = a.means[3 * i], py = a.means[3 * i + 1], pz = a.means[3 * i + 2];
  const float tx = ((W[0] * px + W[1] * py) + W[2] * pz) + W[3];
  const float ty = ((W[4] * px + W[5] * py) + W[6] * pz) + W[7];
  const float tz = ((W[8] * px + W[9] * py) + W[10] * pz) + W[11];
  const float4 q = *reinterpret_cast<const float4*>(a.quats + 4 * i);
  const float w = q.x, x = q.y, y = q.z, z = q.w;
  const float s[3] = {a.scales[3 * i], a.scales[3 * i + 1], a.scales[3 * i + 2]};
  float R[9];
  R[0] = 1.0f - 2.0f * (y * y + z * z); R[1] = 2.0f * (x * y - w * z); R[2] = 2.0f * (x * z + w * y);
  R[3] = 2.0f * (x * y + w * z); R[4] = 1.0f - 2.0f * (x * x + z * z); R[5] = 2.0f * (y * z - w * x);
  R[6] = 2.0f * (x * z - w * y); R[7] = 2.0f * (y * z + w * x); R[8] = 1.0f - 2.0f * (x * x + y * y);
  float M[9];
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) M[3 * r + c] = R[3 * r + c] * s[c];
  float Sg[3][3];
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) Sg[r][c] = (M[3 * r] * M[3 * c] + M[3 * r + 1] * M[3 * c + 1]) + M[3 * r + 2] * M[3 * c + 2];
  const unsigned char cl = a.clamped[i];
  const bool clampx = (cl & 8) != 0, clampy = (cl & 16) != 0;
  const float tanx = (0.5f * (float)cam.width) / cam.fx, tany = (0.5f * (float)cam.height) / cam.fy;
  const float limx = 1.3f * tanx, limy = 1.3f * tany;
  const float xt = fminf(limx, fmaxf(-limx, tx / tz)) * tz, yt = fminf(limy, fmaxf(-limy, ty / tz)) * tz;
  const float tz2 = tz * tz;
  const float J00 = cam.fx / tz, J02 = -((cam.fx * xt) / tz2), J11 = cam.fy / tz, J12 = -((cam.fy * yt) / tz2);
  float Tm[2][3];
#pragma unroll
  for (int k = 0; k < 3; ++k) { Tm[0][k] = J00 * W[k] + J02 * W[8 + k]; Tm[1][k] = J11 * W[4 + k] + J12 * W[8 + k]; }
  // whitened sums -> gradients of opacity, mean2d and the 2D covariance (head of backward.cu):
  //   dL/do = S0 / o;  dL/dmu = R^T (Su, Sv);  dL/dSigma' = 1/2 R^T H R   with R = R' / s, (Su, Sv) = (Su', Sv') / s,
  //   H = H' / s^2, s^2 = log2(e) / 2   =>   dL/dmu = R'^T (Su', Sv') / s^2,  dL/dSigma' = R'^T H' R' / (2 s^4)
  const float4 co = *reinterpret_cast<const float4*>(a.conic_opacity + 4 * i);
  const float* gs = a.gscr + (size_t)i * a.RG;
  const float4 s0 = *reinterpret_cast<const float4*>(gs), s1 = *reinterpret_cast<const float4*>(gs + 4);
  const float* rec = a.record + (size_t)i * a.RS;
  const double r11 = rec[2], r12 = rec[3], r22 = rec[4];
  const double kMu = 1.3862943611198906;     // 1 / s^2   = 2 ln 2
  const double kCov = 0.96090602783640280;   // 1 / (2 s^4) = 2 ln^2 2
  const double Su = s0.y, Sv = s0.z, Huu = s0.w, Huv = s1.x, Hvv = s1.y;
  const float gmx = (float)(kMu * (r11 * Su)), gmy = (float)(kMu * (r12 * Su + r22 * Sv));
  const double m01 = Huu * r12 + Huv * r22, m11 = Huv * r12 + Hvv * r22;
  float Gp[2][2];
  Gp[0][0] = (float)(kCov * (r11 * r11 * Huu));
  Gp[0][1] = (float)(kCov * (r11 * m01));
  Gp[1][0] = Gp[0][1];
  Gp[1][1] = (float)(kCov * (r12 * m01 + r22 * m11));
  store(a.dopac + i, s0.x / co.w, acc);
  const int so = 9 + a.geo;   // first semantic slot
  for (int f = 0; f < a.F; f += 4) {   // F is a multiple of 4: 16-byte stores
    float4* d = reinterpret_cast<float4*>(a.dsem + (size_t)i * a.F + f);
    float4 v = make_float4(gs[so + f], gs[so + f + 1], gs[so + f + 2], gs[so + f + 3]);
    if (acc) { const float4 o = *d; v.x += o.x; v.y += o.y; v.z += o.z; v.w += o.w; }
    *d = v;
  }
  store(a.dunc + i, gs[so + a.F], acc);
  float GT[2][3];
#pragma unroll
  for (int r = 0; r < 2; ++r)
#pragma unroll
    for (int k = 0; k < 3; ++k) GT[r][k] = Gp[r][0] * Tm[0][k] + Gp[r][1] * Tm[1][k];
  float dSig[3][3], dT[2][3];
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int k = 0; k < 3; ++k) dSig[r][k] = Tm[0][r] * GT[0][k] + Tm[1][r] * GT[1][k];
#pragma unroll
  for (int r = 0; r < 2; ++r)
#pragma unroll
    for (int k = 0; k < 3; ++k) dT[r][k] = 2.0f * ((GT[r][0] * Sg[0][k] + GT[r][1] * Sg[1][k]) + GT[r][2] * Sg[2][k]);
  const float dJ00 = (dT[0][0] * W[0] + dT[0][1] * W[1]) + dT[0][2] * W[2];
  const float dJ02 = (dT[0][0] * W[8] + dT[0][1] * W[9]) + dT[0][2] * W[10];
  const float dJ11 = (dT[1][0] * W[4] + dT[1][1] * W[5]) + dT[1][2] * W[6];
  const float dJ12 = (dT[1][0] * W[8] + dT[1][1] * W[9]) + dT[1][2] * W[10];
  float dt0 = 0.f, dt1 = 0.f, dt2 = 0.f;
  if (!clampx) { dt0 += dJ02 * (-cam.fx / tz2); dt2 += dJ02 * ((2.0f * cam.fx * tx) / (tz2 * tz)); }
  else dt2 += dJ02 * (-J02 / tz);
  if (!clampy) { dt1 += dJ12 * (-cam.fy / tz2); dt2 += dJ12 * ((2.0f * cam.fy * ty) / (tz2 * tz)); }
  else dt2 += dJ12 * (-J12 / tz);
  dt2 += dJ00 * (-cam.fx / tz2) + dJ11 * (-cam.fy / tz2);
  dt0 += gmx * (cam.fx / tz);
  dt1 += gmy * (cam.fy / tz);
  dt2 += gmx * (-(cam.fx * tx) / tz2) + gmy * (-(cam.fy * ty) / tz2);
  if (a.geo) dt2 += gs[9];   // the depth image blends t_z itself (LEGS_BWD_DEPTH_ALPHA)
  float dmean[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) dmean[k] = (W[k] * dt0 + W[4 + k] * dt1) + W[8 + k] * dt2;
  // Sigma = M M^T
  float dM[3][3], dR[3][3], dscale[3];
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) dM[r][c] = 2.0f * ((dSig[r][0] * M[c] + dSig[r][1] * M[3 + c]) + dSig[r][2] * M[6 + c]);
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    dscale[c] = (R[c] * dM[0][c] + R[3 + c] * dM[1][c]) + R[6 + c] * dM[2][c];
#pragma unroll
    for (int r = 0; r < 3; ++r) dR[r][c] = dM[r][c] * s[c];
  }
  float dq[4];
  dq[0] = 2.0f * (-z * dR[0][1] + y * dR[0][2] + z * dR[1][0] - x * dR[1][2] - y * dR[2][0] + x * dR[2][1]);
  dq[1] = 2.0f * (y * dR[0][1] + z * dR[0][2] + y * dR[1][0] - 2.0f * x * dR[1][1] - w * dR[1][2] + z * dR[2][0] +
                  w * dR[2][1] - 2.0f * x * dR[2][2]);
  dq[2] = 2.0f * (-2.0f * y * dR[0][0] + x * dR[0][1] + w * dR[0][2] + x * dR[1][0] + z * dR[1][2] - w * dR[2][0] +
                  z * dR[2][1] - 2.0f * y * dR[2][2]);
  dq[3] = 2.0f * (-2.0f * z * dR[0][0] - w * dR[0][1] + x * dR[0][2] + w * dR[1][0] - 2.0f * z * dR[1][1] +
                  y * dR[1][2] + x * dR[2][0] + y * dR[2][1]);
  // colour
  float g3[3];
#pragma unroll
  for (int ch = 0; ch < 3; ++ch) g3[ch] = (cl & (1u << ch)) ? 0.f : gs[6 + ch];
  const float cpx = -((W[0] * W[3] + W[4] * W[7]) + W[8] * W[11]);
  const float cpy = -((W[1] * W[3] + W[5] * W[7]) + W[9] * W[11]);
  const float cpz = -((W[2] * W[3] + W[6] * W[7]) + W[10] * W[11]);
  const float ddx = px - cpx, ddy = py - cpy, ddz = pz - cpz;
  const float len = sqrtf((ddx * ddx + ddy * ddy) + ddz * ddz);
  const float hx = ddx / len, hy = ddy / len, hz = ddz / len;
  float gx = 0.f, gy = 0.f, gz = 0.f;  // dL/d(dhat)
  float ek[16];                         // <c_k, g> for every active coefficient, read before the row is overwritten
  if (BULK) {
    while (!mbar_done(bar, 0)) {}
#pragma unroll
    for (int k = 0; k < 16; ++k) ek[k] = 0.f;
    const int S3 = a.sh_stored * 3;
#pragma unroll
    for (int j = 0; j < 12; ++j) {
      if (4 * j < S3) {
        const float4 v = *reinterpret_cast<const float4*>(srow + 4 * j);
        const float vv[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          const int e = 4 * j + t, k = e / 3, ch = e % 3;
          if (k < nb) ek[k] = ch == 0 ? vv[t] * g3[0] : ek[k] + vv[t] * g3[ch];
        }
      }
    }
  } else {
#pragma unroll
    for (int k = 0; k < 16; ++k)
      ek[k] = k < nb ? (srow[3 * k] * g3[0] + srow[3 * k + 1] * g3[1]) + srow[3 * k + 2] * g3[2] : 0.f;
  }
  auto coef = [&](int k) { return ek[k]; };
  float bas[16];                        // basis values Y_k(dhat): dL/dc_k = Y_k g
#pragma unroll
  for (int k = 0; k < 16; ++k) bas[k] = 0.f;
  auto put = [&](int k, float b) { bas[k] = b; };
  put(0, kC[0]);
  if (a.sh_degree >= 1) {
    put(1, -(kC[1] * hy)); put(2, kC[1] * hz); put(3, -(kC[1] * hx));
    gy += -kC[1] * coef(1); gz += kC[1] * coef(2); gx += -kC[1] * coef(3);
  }
  if (a.sh_degree >= 2) {
    const float xx = hx * hx, yy = hy * hy, zz = hz * hz;
    put(4, kC[2] * (hx * hy)); put(5, -(kC[2] * (hy * hz))); put(6, kC[3] * ((2.0f * zz - xx) - yy));
    put(7, -(kC[2] * (hx * hz))); put(8, kC[4] * (xx - yy));
    const float e4 = coef(4), e5 = coef(5), e6 = coef(6), e7 = coef(7), e8 = coef(8);
    gx += kC[2] * hy * e4 - 2.0f * kC[3] * hx * e6 - kC[2] * hz * e7 + 2.0f * kC[4] * hx * e8;
    gy += kC[2] * hx * e4 - kC[2] * hz * e5 - 2.0f * kC[3] * hy * e6 - 2.0f * kC[4] * hy * e8;
    gz += -kC[2] * hy * e5 + 4.0f * kC[3] * hz * e6 - kC[2] * hx * e7;
    if (a.sh_degree >= 3) {
      put(9, -((kC[5] * hy) * (3.0f * xx - yy)));
      put(10, (kC[6] * (hx * hy)) * hz);
      put(11, -((kC[7] * hy) * ((4.0f * zz - xx) - yy)));
      put(12, (kC[8] * hz) * ((2.0f * zz - 3.0f * xx) - 3.0f * yy));
      put(13, -((kC[7] * hx) * ((4.0f * zz - xx) - yy)));
      put(14, (kC[9] * hz) * (xx - yy));
      put(15, -((kC[5] * hx) * (xx - 3.0f * yy)));
      const float e9 = coef(9), e10 = coef(10), e11 = coef(11), e12 = coef(12), e13 = coef(13), e14 = coef(14), e15 = coef(15);
      gx += -6.0f * kC[5] * hx * hy * e9 + kC[6] * hy * hz * e10 + 2.0f * kC[7] * hx * hy * e11 - 6.0f * kC[8] * hx * hz * e12 -
            kC[7] * (4.0f * zz - 3.0f * xx - yy) * e13 + 2.0f * kC[9] * hx * hz * e14 - kC[5] * (3.0f * xx - 3.0f * yy) * e15;
      gy += -kC[5] * (3.0f * xx - 3.0f * yy) * e9 + kC[6] * hx * hz * e10 - kC[7] * (4.0f * zz - xx - 3.0f * yy) * e11 -
            6.0f * kC[8] * hy * hz * e12 + 2.0f * kC[7] * hx * hy * e13 - 2.0f * kC[9] * hy * hz * e14 + 6.0f * kC[5] * hx * hy * e15;
      gz += kC[6] * hx * hy * e10 - 8.0f * kC[7] * hy * hz * e11 + kC[8] * (6.0f * zz - 3.0f * xx - 3.0f * yy) * e12 -
            8.0f * kC[7] * hx * hz * e13 + kC[9] * (xx - yy) * e14;
    }
  }
  if (BULK) {
    const int S3 = a.sh_stored * 3;
#pragma unroll
    for (int j = 0; j < 12; ++j) {
      if (4 * j < S3) {
        float o[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) o[t] = bas[(4 * j + t) / 3] * g3[(4 * j + t) % 3];
        *reinterpret_cast<float4*>(srow + 4 * j) = make_float4(o[0], o[1], o[2], o[3]);
      }
    }
  } else {
    for (int k = 0; k < a.sh_stored; ++k) {
      const float b = k < 16 ? bas[k < 16 ? k : 0] : 0.f;
      srow[3 * k] = b * g3[0]; srow[3 * k + 1] = b * g3[1]; srow[3 * k + 2] = b * g3[2];
    }
  }
  const float dot = hx * gx + hy * gy + hz * gz;
  dmean[0] += (gx - hx * dot) / len;
  dmean[1] += (gy - hy * dot) / len;
  dmean[2] += (gz - hz * dot) / len;
#pragma unroll
  for (int k = 0; k < 3; ++k) { store(a.dmeans + 3 * i + k, dmean[k], acc); store(a.dscales + 3 * i + k, dscale[k], acc); }
  {
    float4* d = reinterpret_cast<float4*>(a.dquats + 4 * i);
    float4 v = make_float4(dq[0], dq[1], dq[2], dq[3]);
    if (acc) { const float4 o = *d; v.x += o.x; v.y += o.y; v.z += o.z; v.w += o.w; }
    *d = v;
    float2* d2 = reinterpret_cast<float2*>(a.dmean2d + 2 * i);
    float2 v2 = make_float2(gmx, gmy);
    if (acc) { const float2 o = *d2; v2.x += o.x; v2.y += o.y; }
    *d2 = v2;
  }
}

// The SH rows of a block's 128 consecutive Gaussians are one contiguous region of `sh` / `dsh`.
// BULK (sh_stored * 3 a multiple of 4 floats): every visible Gaussian's row comes in by one bulk async copy issued by its
// own thread and its gradient row leaves by one bulk async store (a bulk reduce-add when accumulating): no staging loops,
// rows of culled Gaussians are never read. Otherwise the region is staged through shared memory (pitch S3 | 1).
template <bool BULK>
// 7 CTAs per SM (71 registers, no spills): measured 0.130 -> 0.122 ms against 5 CTAs at 88 registers; 8 CTAs (64) lose again
__global__ void __launch_bounds__(kBlock, 7) project_backward_kernel(PbArgs a, DevCamera cam) {
  extern __shared__ __align__(16) float s_sh[];
  __shared__ unsigned long long s_bar;
  const int S3 = a.sh_stored * 3, pitch = BULK ? (S3 + 4) : (S3 | 1);
  const long long i0 = (long long)blockIdx.x * kBlock;
  const int rows = (int)min((long long)kBlock, a.n - i0);
  const long long i = i0 + threadIdx.x;
  float* srow = s_sh + threadIdx.x * pitch;
  bool live = false;
  if (BULK) {
    if (threadIdx.x == 0) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(&s_bar)), "r"(kBlock));
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    live = i < a.n && a.tiles[i] != 0;
    const unsigned bytes = live ? (unsigned)S3 * 4u : 0u;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(&s_bar)), "r"(bytes) : "memory");
    if (live)
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_addr(srow)),
                   "l"(a.sh + (size_t)i * S3), "r"(bytes), "r"(smem_addr(&s_bar))
                   : "memory");
  } else {
    const float* src = a.sh + (size_t)i0 * S3;
    // (row, column) of element e = threadIdx.x + k * kBlock advanced incrementally: no integer division in the loops
    const int dr = kBlock / S3, dc = kBlock % S3;
    int r = threadIdx.x / S3, c = threadIdx.x % S3;
    for (int e = threadIdx.x; e < rows * S3; e += kBlock) {
      s_sh[r * pitch + c] = src[e];
      r += dr; c += dc;
      if (c >= S3) { c -= S3; ++r; }
    }
    __syncthreads();
    live = i < a.n && a.tiles[i] != 0;
  }
  if (i < a.n) {
    if (!live) {
      if (BULK) {
        if (!a.accumulate)
          for (int k = 0; k < S3; k += 4) *reinterpret_cast<float4*>(srow + k) = make_float4(0.f, 0.f, 0.f, 0.f);
      } else {
        for (int k = 0; k < S3; ++k) srow[k] = 0.f;
      }
      if (!a.accumulate) {
        for (int k = 0; k < 3; ++k) { a.dmeans[3 * i + k] = 0.f; a.dscales[3 * i + k] = 0.f; }
        *reinterpret_cast<float4*>(a.dquats + 4 * i) = make_float4(0.f, 0.f, 0.f, 0.f);
        *reinterpret_cast<float2*>(a.dmean2d + 2 * i) = make_float2(0.f, 0.f);
        a.dopac[i] = 0.f; a.dunc[i] = 0.f;
        for (int f = 0; f < a.F; f += 4) *reinterpret_cast<float4*>(a.dsem + (size_t)i * a.F + f) = make_float4(0.f, 0.f, 0.f, 0.f);
      }
    } else {
      project_backward_one<BULK>(a, cam, i, srow, &s_bar);
    }
  }
  if (BULK) {
    if (i < a.n && (live || !a.accumulate)) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      float* dst = a.dsh + (size_t)i * S3;
      if (a.accumulate)
        asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f32 [%0], [%1], %2;" ::"l"(dst), "r"(smem_addr(srow)),
                     "r"((unsigned)S3 * 4u)
                     : "memory");
      else
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_addr(srow)),
                     "r"((unsigned)S3 * 4u)
                     : "memory");
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    while (!mbar_done(&s_bar, 0)) {}                                   // no inbound copy in flight when the block retires
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");     // the row has left shared memory
    return;
  }
  __syncthreads();
  float* dst = a.dsh + (size_t)i0 * S3;
  const int dr = kBlock / S3, dc = kBlock % S3;
  int r = threadIdx.x / S3, c = threadIdx.x % S3;
  for (int e = threadIdx.x; e < rows * S3; e += kBlock) {
    const float v = s_sh[r * pitch + c];
    dst[e] = a.accumulate ? dst[e] + v : v;
    r += dr; c += dc;
    if (c >= S3) { c -= S3; ++r; }
  }
}

}  // namespace

int legs_project_backward_launch(legs_ctx* ctx, const legs_gaussians* g, const DevCamera& dc, const legs_frame* frame,
                                 const float* gscr, legs_grads* grads, int accumulate, int geo, cudaStream_t st) {
  PbArgs a;
  a.n = g->n; a.sh_degree = g->sh_degree; a.sh_stored = g->sh_coefs_stored; a.accumulate = accumulate;
  a.means = g->means; a.scales = g->scales; a.quats = g->quats; a.sh = g->sh;
  a.tiles = frame->tiles_touched; a.clamped = frame->clamped; a.conic_opacity = frame->conic_opacity;
  a.F = g->sem_dim; a.RS = legs_record_stride(g->sem_dim); a.geo = geo ? 1 : 0;
  a.RG = (6 + (g->sem_dim + 4 + a.geo + 3) / 4 * 4 + 3) / 4 * 4;
  a.record = frame->record; a.gscr = gscr;
  a.dmeans = grads->dmeans; a.dscales = grads->dscales; a.dquats = grads->dquats; a.dsh = grads->dsh;
  a.dmean2d = grads->dmean2d; a.dopac = grads->dopacities; a.dsem = grads->dsem; a.dunc = grads->dunc;
  const int nb = (int)((g->n + kBlock - 1) / kBlock);
  const int S3 = a.sh_stored * 3;
  const bool bulk = (S3 % 4) == 0 && S3 <= 48 && legs_aligned16(a.sh) && legs_aligned16(a.dsh);
  const size_t smem = (size_t)kBlock * (bulk ? (S3 + 4) : (S3 | 1)) * sizeof(float);
  if (bulk) project_backward_kernel<true><<<nb, kBlock, smem, st>>>(a, dc);
  else project_backward_kernel<false><<<nb, kBlock, smem, st>>>(a, dc);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

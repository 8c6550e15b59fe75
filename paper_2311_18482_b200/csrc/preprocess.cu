// preprocess.cu — S1: per-Gaussian projection (DESIGN.md "Forward, per Gaussian" steps 1-8) and D = sum tiles_touched.
//
// Rule P-0: this translation unit is compiled with --fmad=false -prec-div=true -prec-sqrt=true -ftz=false so that
// every written operation is one IEEE binary32 rounding; integer results (radius, rect, tiles_touched, depth bits)
// are then reproducible bit for bit. The kernel is HBM-bound, so the un-fused arithmetic is free.
//
// PAPER.md:56-58 (Eq. 1) names the attributes; the projection maths is the EWA reading C-1..C-12.
#include "common.cuh"

namespace {

constexpr int kBlock = 128;

// Real spherical-harmonic normalisation constants (Condon-Shortley sign), 17 significant digits.
__device__ __constant__ float kSH[10] = {
    0.28209479177387814f,  // 1/2 sqrt(1/pi)
    0.48860251190291992f,  // sqrt(3/(4 pi))
    1.0925484305920792f,   // 1/2 sqrt(15/pi)
    0.31539156525252005f,  // 1/4 sqrt(5/pi)
    0.54627421529603959f,  // 1/4 sqrt(15/pi)
    0.59004358992664352f,  // 1/4 sqrt(35/(2 pi))
    2.8906114426405538f,   // 1/2 sqrt(105/pi)
    0.45704579946446572f,  // 1/4 sqrt(21/(2 pi))
    0.37317633259011540f,  // 1/4 sqrt(7/pi)
    1.4453057213202769f    // 1/4 sqrt(105/pi)
};

__device__ __forceinline__ void eval_sh_basis(float x, float y, float z, int degree, float* b) {
  b[0] = kSH[0];
  if (degree < 1) return;
  b[1] = -(kSH[1] * y);
  b[2] = kSH[1] * z;
  b[3] = -(kSH[1] * x);
  if (degree < 2) return;
  const float xx = x * x, yy = y * y, zz = z * z, xy = x * y, yz = y * z, xz = x * z;
  b[4] = kSH[2] * xy;
  b[5] = -(kSH[2] * yz);
  b[6] = kSH[3] * ((2.0f * zz - xx) - yy);
  b[7] = -(kSH[2] * xz);
  b[8] = kSH[4] * (xx - yy);
  if (degree < 3) return;
  b[9] = -((kSH[5] * y) * (3.0f * xx - yy));
  b[10] = (kSH[6] * xy) * z;
  b[11] = -((kSH[7] * y) * ((4.0f * zz - xx) - yy));
  b[12] = (kSH[8] * z) * ((2.0f * zz - 3.0f * xx) - 3.0f * yy);
  b[13] = -((kSH[7] * x) * ((4.0f * zz - xx) - yy));
  b[14] = (kSH[9] * z) * (xx - yy);
  b[15] = -((kSH[5] * x) * (xx - 3.0f * yy));
}

struct PreArgs {
  long long n;
  int sh_degree, sh_stored, F, RS;
  const float *means, *scales, *quats, *opac, *sh, *sem, *unc;
  float* depth; int* radius; int* rect; float* mean2d; float* conic_opacity; float* rgb; unsigned char* clamped;
  unsigned int* tiles; float* record;
  unsigned long long* num_instances;
};

// mbarrier + bulk async copy (TMA without a tensor map), local copies of the two wrappers this file needs
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ bool mbar_done(unsigned long long* bar, unsigned parity) {
  unsigned ok;
  asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(ok) : "r"(smem_addr(bar)), "r"(parity) : "memory");
  return ok != 0;
}

// BULK: sh_stored * 3 is a multiple of 4 floats (16 coefficients: 192 B per Gaussian), so every thread fetches its own SH
// row with ONE bulk async copy, issued as soon as the near-plane test has passed and waited for only when the colour is
// evaluated: no staging loop, the copy overlaps the projection arithmetic, and culled Gaussians never read their row.
// Rows sit at a pitch of an odd number of 16-byte units, so the per-thread float4 row reads are conflict-free.
template <bool BULK>
__global__ void __launch_bounds__(kBlock) preprocess_kernel(PreArgs a, DevCamera cam) {
  extern __shared__ __align__(16) float s_sh[];
  __shared__ unsigned long long s_bar;
  const int S3 = a.sh_stored * 3, pitch = BULK ? (S3 + 4) : (S3 | 1);
  if (BULK) {
    if (threadIdx.x == 0) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(&s_bar)), "r"(kBlock));
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
  } else {
    // the SH rows of the block's consecutive Gaussians are one contiguous region: staged through shared memory with
    // coalesced loads (pitch S3 | 1: odd, so the per-thread row reads are conflict-free)
    const long long i0 = (long long)blockIdx.x * kBlock;
    const int rows = (int)min((long long)kBlock, a.n - i0);
    const float* src = a.sh + (size_t)i0 * S3;
    // (row, column) of element e = threadIdx.x + k * kBlock advanced incrementally: no integer division in the loop
    const int dr = kBlock / S3, dc = kBlock % S3;
    int r = threadIdx.x / S3, c = threadIdx.x % S3;
    for (int e = threadIdx.x; e < rows * S3; e += kBlock) {
      s_sh[r * pitch + c] = src[e];
      r += dr; c += dc;
      if (c >= S3) { c -= S3; ++r; }
    }
    __syncthreads();
  }
  const long long i = (long long)blockIdx.x * kBlock + threadIdx.x;
  unsigned int tiles = 0;
  if (i < a.n) {
    const float px = a.means[3 * i], py = a.means[3 * i + 1], pz = a.means[3 * i + 2];
    const float* W = cam.W;
    const float tx = ((W[0] * px + W[1] * py) + W[2] * pz) + W[3];
    const float ty = ((W[4] * px + W[5] * py) + W[6] * pz) + W[7];
    const float tz = ((W[8] * px + W[9] * py) + W[10] * pz) + W[11];
    int rad = 0, x0 = 0, y0 = 0, x1 = 0, y1 = 0;
    float mux = 0.f, muy = 0.f, cA = 0.f, cB = 0.f, cC = 0.f, op = 0.f, cr = 0.f, cg = 0.f, cb = 0.f;
    unsigned char clampbits = 0;
    bool vis = tz > cam.near_plane;
    if (BULK) {
      // every thread arrives once; a Gaussian in front of the near plane also announces and fetches its row
      const unsigned bytes = vis ? (unsigned)S3 * 4u : 0u;
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(&s_bar)), "r"(bytes) : "memory");
      if (vis)
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                         smem_addr(s_sh + threadIdx.x * pitch)),
                     "l"(a.sh + (size_t)i * S3), "r"(bytes), "r"(smem_addr(&s_bar))
                     : "memory");
    }
    if (vis) {
      const float4 q = *reinterpret_cast<const float4*>(a.quats + 4 * i);
      const float w = q.x, x = q.y, y = q.z, z = q.w;
      const float sx = a.scales[3 * i], sy = a.scales[3 * i + 1], sz = a.scales[3 * i + 2];
      const float R00 = 1.0f - 2.0f * (y * y + z * z), R01 = 2.0f * (x * y - w * z), R02 = 2.0f * (x * z + w * y);
      const float R10 = 2.0f * (x * y + w * z), R11 = 1.0f - 2.0f * (x * x + z * z), R12 = 2.0f * (y * z - w * x);
      const float R20 = 2.0f * (x * z - w * y), R21 = 2.0f * (y * z + w * x), R22 = 1.0f - 2.0f * (x * x + y * y);
      const float M00 = R00 * sx, M01 = R01 * sy, M02 = R02 * sz;
      const float M10 = R10 * sx, M11 = R11 * sy, M12 = R12 * sz;
      const float M20 = R20 * sx, M21 = R21 * sy, M22 = R22 * sz;
      const float S00 = (M00 * M00 + M01 * M01) + M02 * M02;
      const float S01 = (M00 * M10 + M01 * M11) + M02 * M12;
      const float S02 = (M00 * M20 + M01 * M21) + M02 * M22;
      const float S11 = (M10 * M10 + M11 * M11) + M12 * M12;
      const float S12 = (M10 * M20 + M11 * M21) + M12 * M22;
      const float S22 = (M20 * M20 + M21 * M21) + M22 * M22;
      const float tanx = (0.5f * (float)cam.width) / cam.fx, tany = (0.5f * (float)cam.height) / cam.fy;
      const float limx = 1.3f * tanx, limy = 1.3f * tany;
      const float xz = tx / tz, yz = ty / tz;
      if (xz < -limx || xz > limx) clampbits |= 8;
      if (yz < -limy || yz > limy) clampbits |= 16;
      const float xt = fminf(limx, fmaxf(-limx, xz)) * tz;
      const float yt = fminf(limy, fmaxf(-limy, yz)) * tz;
      const float J00 = cam.fx / tz, J02 = -((cam.fx * xt) / (tz * tz));
      const float J11 = cam.fy / tz, J12 = -((cam.fy * yt) / (tz * tz));
      const float T00 = J00 * W[0] + J02 * W[8], T01 = J00 * W[1] + J02 * W[9], T02 = J00 * W[2] + J02 * W[10];
      const float T10 = J11 * W[4] + J12 * W[8], T11 = J11 * W[5] + J12 * W[9], T12 = J11 * W[6] + J12 * W[10];
      const float V00 = (T00 * S00 + T01 * S01) + T02 * S02;
      const float V01 = (T00 * S01 + T01 * S11) + T02 * S12;
      const float V02 = (T00 * S02 + T01 * S12) + T02 * S22;
      const float V10 = (T10 * S00 + T11 * S01) + T12 * S02;
      const float V11 = (T10 * S01 + T11 * S11) + T12 * S12;
      const float V12 = (T10 * S02 + T11 * S12) + T12 * S22;
      const float c00 = (V00 * T00 + V01 * T01) + V02 * T02;
      const float c01 = (V00 * T10 + V01 * T11) + V02 * T12;
      const float c11 = (V10 * T10 + V11 * T11) + V12 * T12;
      const float ca = c00 + 0.3f, cbb = c01, cc = c11 + 0.3f;
      const float det = ca * cc - cbb * cbb;
      vis = (det > 0.0f) && isfinite(det);
      if (vis) {
        cA = cc / det;
        cB = (-cbb) / det;
        cC = ca / det;
        const float mid = 0.5f * (ca + cc);
        const float lam = mid + sqrtf(fmaxf(0.1f, mid * mid - det));
        const float rfull = ceilf(3.0f * sqrtf(lam));
        mux = (cam.fx * tx) / tz + (cam.cx - 0.5f);
        muy = (cam.fy * ty) / tz + (cam.cy - 0.5f);
        vis = isfinite(rfull) && isfinite(mux) && isfinite(muy);
        if (vis) {
          const float rf = fminf(rfull, 1073741824.0f);
          rad = (int)rf;
          const float Gx = (float)cam.grid_x, Gy = (float)cam.grid_y;
          x0 = (int)fminf(Gx, fmaxf(0.0f, floorf((mux - rf) / 16.0f)));
          y0 = (int)fminf(Gy, fmaxf(0.0f, floorf((muy - rf) / 16.0f)));
          x1 = (int)fminf(Gx, fmaxf(0.0f, floorf(((mux + rf) + 15.0f) / 16.0f)));
          y1 = (int)fminf(Gy, fmaxf(0.0f, floorf(((muy + rf) + 15.0f) / 16.0f)));
          vis = (x1 - x0) > 0 && (y1 - y0) > 0;
        }
      }
      if (vis) {
        tiles = (unsigned int)(x1 - x0) * (unsigned int)(y1 - y0);
        op = a.opac[i];
        // colour: SH evaluated in the direction camera centre -> mean
        const float cpx = -((W[0] * W[3] + W[4] * W[7]) + W[8] * W[11]);
        const float cpy = -((W[1] * W[3] + W[5] * W[7]) + W[9] * W[11]);
        const float cpz = -((W[2] * W[3] + W[6] * W[7]) + W[10] * W[11]);
        const float dx = px - cpx, dy = py - cpy, dz = pz - cpz;
        const float len = sqrtf((dx * dx + dy * dy) + dz * dz);
        float b[16];
        eval_sh_basis(dx / len, dy / len, dz / len, a.sh_degree, b);
        const int nb = (a.sh_degree + 1) * (a.sh_degree + 1);
        const float* c = s_sh + threadIdx.x * pitch;
        if (BULK) { while (!mbar_done(&s_bar, 0)) {} }
        float acc0 = 0.f, acc1 = 0.f, acc2 = 0.f;
        if (BULK) {
          // the same sums in the same order (k ascending per channel), read as 16-byte chunks of the row
#pragma unroll
          for (int j = 0; j < 12; ++j) {
            if (4 * j < S3) {
              const float4 v = *reinterpret_cast<const float4*>(c + 4 * j);
              const float vv[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
              for (int t = 0; t < 4; ++t) {
                const int e = 4 * j + t, k = e / 3, ch = e % 3;
                if (k < nb) {
                  float& A = ch == 0 ? acc0 : (ch == 1 ? acc1 : acc2);
                  A = (k == 0) ? b[0] * vv[t] : A + b[k] * vv[t];
                }
              }
            }
          }
        } else {
          acc0 = b[0] * c[0]; acc1 = b[0] * c[1]; acc2 = b[0] * c[2];
          for (int k = 1; k < nb; ++k) {
            acc0 = acc0 + b[k] * c[3 * k];
            acc1 = acc1 + b[k] * c[3 * k + 1];
            acc2 = acc2 + b[k] * c[3 * k + 2];
          }
        }
        acc0 = acc0 + 0.5f; acc1 = acc1 + 0.5f; acc2 = acc2 + 0.5f;
        if (acc0 < 0.0f) { clampbits |= 1; acc0 = 0.0f; }
        if (acc1 < 0.0f) { clampbits |= 2; acc1 = 0.0f; }
        if (acc2 < 0.0f) { clampbits |= 4; acc2 = 0.0f; }
        cr = acc0; cg = acc1; cb = acc2;
      } else {
        rad = 0; x0 = y0 = x1 = y1 = 0; mux = muy = 0.f; cA = cB = cC = 0.f; clampbits = 0;
      }
    }
    a.depth[i] = tz;
    a.radius[i] = rad;
    *reinterpret_cast<int4*>(a.rect + 4 * i) = make_int4(x0, y0, x1, y1);
    *reinterpret_cast<float2*>(a.mean2d + 2 * i) = make_float2(mux, muy);
    *reinterpret_cast<float4*>(a.conic_opacity + 4 * i) = make_float4(cA, cB, cC, op);
    a.rgb[3 * i] = cr; a.rgb[3 * i + 1] = cg; a.rgb[3 * i + 2] = cb;
    a.clamped[i] = clampbits;
    a.tiles[i] = tiles;
    if (vis) {
      float* r = a.record + (size_t)i * a.RS;
      // The compositors evaluate the exponent through the Cholesky factor of the conic, Q = R^T R, R upper triangular:
      // d^T Q d = u^2 + v^2 with u = r11 dx + r12 dy, v = r22 dy -- a sum of two squares (no cancellation between
      // A dx^2, C dy^2 and 2 B dx dy for elongated footprints) in one instruction less. R is taken in fp64 from the
      // fp32 conic (r22^2 = (AC - B^2)/A cancels in fp32) and scaled by sqrt(log2(e)/2), so that
      // exp(-d^T Q d / 2) = 2^-(u'^2 + v'^2). A conic that is not positive definite after its fp32 rounding
      // (a c / det beyond ~4e6) gets r22 = 0.
      const double r11 = sqrt((double)cA), r12 = (double)cB / r11;
      const double rem = (double)cC - r12 * r12;
      const double r22 = rem > 0.0 ? sqrt(rem) : 0.0;
      const double kS = 0.84932180028801907;   // sqrt(log2(e) / 2)
      const float w11 = (float)(kS * r11), w12 = (float)(kS * r12), w22 = (float)(kS * r22);
      const bool wok = isfinite(w11) && isfinite(w12) && isfinite(w22);
      reinterpret_cast<float4*>(r)[0] = make_float4(mux, muy, wok ? w11 : 0.f, wok ? w12 : 0.f);
      reinterpret_cast<float4*>(r)[1] = make_float4(wok ? w22 : 0.f, op, cr, cg);
      const float* s = a.sem + (size_t)i * a.F;
      // slots: 8 = b, 9 = depth, 10.. = sem[F], 10+F = u, rest pad
      float tail[2 + LEGS_MAX_SEM_DIM + 4];
      tail[0] = cb; tail[1] = tz;
      for (int f = 0; f < a.F; f += 4) {
        const float4 v = *reinterpret_cast<const float4*>(s + f);
        tail[2 + f] = v.x; tail[3 + f] = v.y; tail[4 + f] = v.z; tail[5 + f] = v.w;
      }
      tail[2 + a.F] = a.unc[i];
      for (int k = 3 + a.F; k < a.RS - 8; ++k) tail[k] = 0.f;
      // last slot: cull threshold of the compositors, in the scaled units of the record: alpha = o 2^-q' >= 1/255 needs
      // q' = u'^2 + v'^2 <= log2(255 o); a little margin on top (the compositors add the rounding bound of their own
      // evaluation of q'). Negative when o < 1/255 (such a Gaussian never passes the alpha test) or R is not finite.
      {
        const float L = log2f(255.0f * op);
        tail[a.RS - 9] = (L >= 0.0f && wok) ? L * 1.001f + 0.015f : -1.0f;
      }
      for (int k = 0; k < a.RS - 8; k += 4)
        reinterpret_cast<float4*>(r + 8)[k / 4] = make_float4(tail[k], tail[k + 1], tail[k + 2], tail[k + 3]);
    }
  }
  else if (BULK) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(&s_bar)) : "memory");
  }
  // block sum of tiles_touched for the scan
  __shared__ unsigned int warp_sums[kBlock / 32];
  if (BULK) { while (!mbar_done(&s_bar, 0)) {} }   // no copy may be in flight when the block retires
  unsigned int v = tiles;
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) warp_sums[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long s = 0;
    for (int k = 0; k < kBlock / 32; ++k) s += warp_sums[k];
    if (s) atomicAdd(a.num_instances, s);
  }
}

}  // namespace

extern "C" {

int32_t legs_record_stride(int32_t F) { return (11 + F + 3) / 4 * 4; }
int32_t legs_pixel_channels(int32_t F) { return (3 + 1 + F + 1 + 1 + 3) / 4 * 4; }

int legs_preprocess(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam, legs_frame* frame, void* stream) {
  if (!ctx) return LEGS_ERR_NULL;
  int rc;
  if ((rc = legs_check_gaussians(g)) != LEGS_OK) return rc;
  if ((rc = legs_check_camera(cam)) != LEGS_OK) return rc;
  if ((rc = legs_check_frame(frame)) != LEGS_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  LEGS_CUDA_CHECK(ctx, cudaMemsetAsync(frame->num_instances, 0, sizeof(uint64_t), st));
  if (g->n == 0) return LEGS_OK;
  PreArgs a;
  a.n = g->n; a.sh_degree = g->sh_degree; a.sh_stored = g->sh_coefs_stored; a.F = g->sem_dim;
  a.RS = legs_record_stride(g->sem_dim);
  a.means = g->means; a.scales = g->scales; a.quats = g->quats; a.opac = g->opacities; a.sh = g->sh; a.sem = g->sem;
  a.unc = g->unc;
  a.depth = frame->depth; a.radius = frame->radius; a.rect = frame->rect; a.mean2d = frame->mean2d;
  a.conic_opacity = frame->conic_opacity; a.rgb = frame->rgb; a.clamped = frame->clamped; a.tiles = frame->tiles_touched;
  a.record = frame->record;
  a.num_instances = (unsigned long long*)frame->num_instances;
  const DevCamera dc = make_dev_camera(cam);
  const int nb = (int)((g->n + kBlock - 1) / kBlock);
  const int S3 = a.sh_stored * 3;
  const bool bulk = (S3 % 4) == 0 && S3 <= 48 && legs_aligned16(a.sh);
  const size_t smem = (size_t)kBlock * (bulk ? (S3 + 4) : (S3 | 1)) * sizeof(float);
  if (bulk) preprocess_kernel<true><<<nb, kBlock, smem, st>>>(a, dc);
  else preprocess_kernel<false><<<nb, kBlock, smem, st>>>(a, dc);
  LEGS_LAUNCH_CHECK(ctx);
  return LEGS_OK;
}

int legs_read_num_instances(legs_ctx* ctx, const legs_frame* frame, uint64_t* host_out, void* stream) {
  if (!ctx || !frame || !frame->num_instances || !host_out) return LEGS_ERR_NULL;
  cudaStream_t st = (cudaStream_t)stream;
  uint64_t v = 0;
  LEGS_CUDA_CHECK(ctx, cudaMemcpyAsync(&v, frame->num_instances, sizeof(v), cudaMemcpyDeviceToHost, st));
  LEGS_CUDA_CHECK(ctx, cudaStreamSynchronize(st));
  *host_out = v & ~LEGS_OVERFLOW_BIT;
  return (v & LEGS_OVERFLOW_BIT) ? LEGS_ERR_CAPACITY : LEGS_OK;
}

}  // extern "C"

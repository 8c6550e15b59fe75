// legs_oracle.cpp — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct CPU oracle for the hot path of "Language Embedded 3D Gaussians"
// (arxiv 2311.18482): rasterisation R, R_s, R_u (PAPER.md:56-58 Eq. 1; :116-122 Eq. 8; :138 Eq. 10),
// its reverse-mode gradients (PAPER.md:56 "differentiable rendering", :182), and the per-pixel codebook
// decode (Eq. 21-22, Table 3) with the relevancy cosine.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call this.
// It shares no code, header, table or constant with the CUDA path (paper_2311_18482_b200/csrc, include/).
//
// The paper delegates all rasteriser mathematics to its reference [17] ("incorporate the CUDA
// kernel from [17]") which is not available; the definition implemented here is the EWA-splatting reading
// listed in DESIGN.md "Readings" (C-1..C-17). Structure, by design of the oracle:
//   * one loop over Gaussians (projection),
//   * one global sort by (depth bits, index),
//   * for each pixel ONE walk over that global list with the membership test tile(pixel) in rect(g)
//     (no tile lists, no batching, no shared memory analogue),
//   * gradients by textbook reverse-mode over the recorded per-pixel contributor list,
//   * decode as naive matrix products in fp64.
//
// Arithmetic: mode 0 = rule P-0 (projection in IEEE binary32, one rounding per written operation, no FMA
// contraction: compile with -ffp-contract=off, never -ffast-math), results widened to fp64 for compositing
// and gradients. mode 1 = everything in fp64 (used for finite differences only).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): closed-form isotropic projection, alpha = o*exp(-1/2 d^T S^-1 d),
// sum(w) + T_final = 1, T monotone, R_u in [0,1], permutation invariance, SH Gram matrix = I by quadrature,
// brute-force tile lists, central finite differences, isolation-flag identities, decode vs one-hot (Eq. 3),
// softmax rows sum to 1, relevancy = 1 for a matching query, Gram shortcut. No function here is "parity unpinned".

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <numeric>
#include <vector>

namespace {

// ---------------------------------------------------------------------------------------------------
// Per-Gaussian projection (steps 1-8 of DESIGN.md "Forward, per Gaussian"), templated on the scalar type.

template <class T>
struct Cam {
  T fx, fy, cx, cy;
  T W[12];  // row-major 3x4 [R|t]
  T near_plane;
  int width, height;
};

template <class T>
struct Proj {
  bool visible;
  T t[3];          // view-space position
  T R[9];          // rotation from quaternion
  T M[9];          // R * diag(s)
  T Sig[6];        // 3D covariance: 00 01 02 11 12 22
  T xt, yt;        // clamped t_x, t_y used in the Jacobian
  bool clampx, clampy;
  T J00, J02, J11, J12;
  T Tm[6];         // T = J * R_wc (2x3): T00 T01 T02 T10 T11 T12
  T a, b, c, det;  // dilated 2D covariance and its determinant
  T A, B, C;       // conic
  T mu[2];
  T radius_f;
  int radius;
  int rect[4];
  uint32_t tiles;
  T dir[3], dirlen, dhat[3];
  T basis[16];
  T rgb_raw[3];    // before clamp at 0 (includes +0.5)
  T rgb[3];
  uint8_t clamped; // bit0..2 rgb<0, bit3/4 Jacobian x/y clamp
};

// Real SH basis constants from their closed forms (Condon-Shortley sign convention).
template <class T>
struct SHC {
  T c0, c1, c2a, c2b, c2c, c3a, c3b, c3c, c3d, c3e;
  SHC() {
    const double pi = 3.14159265358979323846;
    c0 = (T)(0.5 * std::sqrt(1.0 / pi));
    c1 = (T)(std::sqrt(3.0 / (4.0 * pi)));
    c2a = (T)(0.5 * std::sqrt(15.0 / pi));
    c2b = (T)(0.25 * std::sqrt(5.0 / pi));
    c2c = (T)(0.25 * std::sqrt(15.0 / pi));
    c3a = (T)(0.25 * std::sqrt(35.0 / (2.0 * pi)));
    c3b = (T)(0.5 * std::sqrt(105.0 / pi));
    c3c = (T)(0.25 * std::sqrt(21.0 / (2.0 * pi)));
    c3d = (T)(0.25 * std::sqrt(7.0 / pi));
    c3e = (T)(0.25 * std::sqrt(105.0 / pi));
  }
};

template <class T>
void sh_basis(const T d[3], int degree, T* b) {
  static const SHC<T> k;
  const T x = d[0], y = d[1], z = d[2];
  b[0] = k.c0;
  if (degree < 1) return;
  b[1] = -(k.c1 * y);
  b[2] = k.c1 * z;
  b[3] = -(k.c1 * x);
  if (degree < 2) return;
  const T xx = x * x, yy = y * y, zz = z * z, xy = x * y, yz = y * z, xz = x * z;
  b[4] = k.c2a * xy;
  b[5] = -(k.c2a * yz);
  b[6] = k.c2b * (((T)2 * zz - xx) - yy);
  b[7] = -(k.c2a * xz);
  b[8] = k.c2c * (xx - yy);
  if (degree < 3) return;
  b[9] = -((k.c3a * y) * ((T)3 * xx - yy));
  b[10] = (k.c3b * xy) * z;
  b[11] = -((k.c3c * y) * (((T)4 * zz - xx) - yy));
  b[12] = (k.c3d * z) * (((T)2 * zz - (T)3 * xx) - (T)3 * yy);
  b[13] = -((k.c3c * x) * (((T)4 * zz - xx) - yy));
  b[14] = (k.c3e * z) * (xx - yy);
  b[15] = -((k.c3a * x) * (xx - (T)3 * yy));
}

// Gradient of each basis function with respect to the (unit) direction, treating x,y,z as free variables.
template <class T>
void sh_basis_grad(const T d[3], int degree, T (*g)[3]) {
  static const SHC<T> k;
  const T x = d[0], y = d[1], z = d[2];
  for (int i = 0; i < 16; ++i) g[i][0] = g[i][1] = g[i][2] = (T)0;
  if (degree < 1) return;
  g[1][1] = -k.c1;
  g[2][2] = k.c1;
  g[3][0] = -k.c1;
  if (degree < 2) return;
  g[4][0] = k.c2a * y;  g[4][1] = k.c2a * x;
  g[5][1] = -k.c2a * z; g[5][2] = -k.c2a * y;
  g[6][0] = -(T)2 * k.c2b * x; g[6][1] = -(T)2 * k.c2b * y; g[6][2] = (T)4 * k.c2b * z;
  g[7][0] = -k.c2a * z; g[7][2] = -k.c2a * x;
  g[8][0] = (T)2 * k.c2c * x; g[8][1] = -(T)2 * k.c2c * y;
  if (degree < 3) return;
  const T xx = x * x, yy = y * y, zz = z * z;
  // b9 = -c3a*y*(3xx - yy)
  g[9][0] = -k.c3a * y * (T)6 * x;  g[9][1] = -k.c3a * ((T)3 * xx - (T)3 * yy);
  // b10 = c3b*x*y*z
  g[10][0] = k.c3b * y * z; g[10][1] = k.c3b * x * z; g[10][2] = k.c3b * x * y;
  // b11 = -c3c*y*(4zz - xx - yy)
  g[11][0] = k.c3c * y * (T)2 * x; g[11][1] = -k.c3c * ((T)4 * zz - xx - (T)3 * yy); g[11][2] = -k.c3c * y * (T)8 * z;
  // b12 = c3d*z*(2zz - 3xx - 3yy)
  g[12][0] = -k.c3d * z * (T)6 * x; g[12][1] = -k.c3d * z * (T)6 * y; g[12][2] = k.c3d * ((T)6 * zz - (T)3 * xx - (T)3 * yy);
  // b13 = -c3c*x*(4zz - xx - yy)
  g[13][0] = -k.c3c * ((T)4 * zz - (T)3 * xx - yy); g[13][1] = k.c3c * x * (T)2 * y; g[13][2] = -k.c3c * x * (T)8 * z;
  // b14 = c3e*z*(xx - yy)
  g[14][0] = k.c3e * z * (T)2 * x; g[14][1] = -k.c3e * z * (T)2 * y; g[14][2] = k.c3e * (xx - yy);
  // b15 = -c3a*x*(xx - 3yy)
  g[15][0] = -k.c3a * ((T)3 * xx - (T)3 * yy); g[15][1] = k.c3a * x * (T)6 * y;
}

template <class T>
inline bool finite_t(T v) { return std::isfinite(v); }

template <class T>
void project_one(const T p[3], const T s[3], const T q[4], const T* sh /*[stored,3]*/, int sh_degree,
                 const Cam<T>& cam, Proj<T>& o) {
  o.visible = false;
  o.tiles = 0;
  o.radius = 0;
  o.rect[0] = o.rect[1] = o.rect[2] = o.rect[3] = 0;
  o.clamped = 0;
  const T* W = cam.W;
  // 1. view transform
  o.t[0] = ((W[0] * p[0] + W[1] * p[1]) + W[2] * p[2]) + W[3];
  o.t[1] = ((W[4] * p[0] + W[5] * p[1]) + W[6] * p[2]) + W[7];
  o.t[2] = ((W[8] * p[0] + W[9] * p[1]) + W[10] * p[2]) + W[11];
  const T tx = o.t[0], ty = o.t[1], tz = o.t[2];
  if (!(tz > cam.near_plane)) return;  // near cull (also rejects NaN)
  // 2. 3D covariance from scale + quaternion (w,x,y,z), no normalisation inside
  const T w = q[0], x = q[1], y = q[2], z = q[3];
  T* R = o.R;
  R[0] = (T)1 - (T)2 * (y * y + z * z); R[1] = (T)2 * (x * y - w * z);         R[2] = (T)2 * (x * z + w * y);
  R[3] = (T)2 * (x * y + w * z);         R[4] = (T)1 - (T)2 * (x * x + z * z); R[5] = (T)2 * (y * z - w * x);
  R[6] = (T)2 * (x * z - w * y);         R[7] = (T)2 * (y * z + w * x);         R[8] = (T)1 - (T)2 * (x * x + y * y);
  T* M = o.M;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) M[3 * i + j] = R[3 * i + j] * s[j];
  auto sig = [&](int i, int j) { return (M[3 * i] * M[3 * j] + M[3 * i + 1] * M[3 * j + 1]) + M[3 * i + 2] * M[3 * j + 2]; };
  o.Sig[0] = sig(0, 0); o.Sig[1] = sig(0, 1); o.Sig[2] = sig(0, 2);
  o.Sig[3] = sig(1, 1); o.Sig[4] = sig(1, 2); o.Sig[5] = sig(2, 2);
  // 3. Jacobian with the 1.3 x tan(half-fov) clamp
  const T tanx = ((T)0.5 * (T)cam.width) / cam.fx, tany = ((T)0.5 * (T)cam.height) / cam.fy;
  const T limx = (T)1.3 * tanx, limy = (T)1.3 * tany;
  const T xz = tx / tz, yz = ty / tz;
  o.clampx = (xz < -limx) || (xz > limx);
  o.clampy = (yz < -limy) || (yz > limy);
  const T cxz = std::min(limx, std::max(-limx, xz)), cyz = std::min(limy, std::max(-limy, yz));
  o.xt = cxz * tz;
  o.yt = cyz * tz;
  o.J00 = cam.fx / tz;
  o.J02 = -((cam.fx * o.xt) / (tz * tz));
  o.J11 = cam.fy / tz;
  o.J12 = -((cam.fy * o.yt) / (tz * tz));
  T* Tm = o.Tm;
  for (int k = 0; k < 3; ++k) {
    Tm[k] = o.J00 * W[k] + o.J02 * W[8 + k];
    Tm[3 + k] = o.J11 * W[4 + k] + o.J12 * W[8 + k];
  }
  const T S00 = o.Sig[0], S01 = o.Sig[1], S02 = o.Sig[2], S11 = o.Sig[3], S12 = o.Sig[4], S22 = o.Sig[5];
  const T V00 = (Tm[0] * S00 + Tm[1] * S01) + Tm[2] * S02;
  const T V01 = (Tm[0] * S01 + Tm[1] * S11) + Tm[2] * S12;
  const T V02 = (Tm[0] * S02 + Tm[1] * S12) + Tm[2] * S22;
  const T V10 = (Tm[3] * S00 + Tm[4] * S01) + Tm[5] * S02;
  const T V11 = (Tm[3] * S01 + Tm[4] * S11) + Tm[5] * S12;
  const T V12 = (Tm[3] * S02 + Tm[4] * S12) + Tm[5] * S22;
  const T c00 = (V00 * Tm[0] + V01 * Tm[1]) + V02 * Tm[2];
  const T c01 = (V00 * Tm[3] + V01 * Tm[4]) + V02 * Tm[5];
  const T c11 = (V10 * Tm[3] + V11 * Tm[4]) + V12 * Tm[5];
  // 4. dilation, determinant, conic
  o.a = c00 + (T)0.3;
  o.b = c01;
  o.c = c11 + (T)0.3;
  o.det = o.a * o.c - o.b * o.b;
  if (!(o.det > (T)0) || !finite_t(o.det)) return;
  o.A = o.c / o.det;
  o.B = (-o.b) / o.det;
  o.C = o.a / o.det;
  // 5. radius
  const T mid = (T)0.5 * (o.a + o.c);
  const T lam = mid + std::sqrt(std::max((T)0.1, mid * mid - o.det));
  o.radius_f = std::ceil((T)3 * std::sqrt(lam));
  // 6. pixel-index-space mean (unclamped t)
  o.mu[0] = (cam.fx * tx) / tz + (cam.cx - (T)0.5);
  o.mu[1] = (cam.fy * ty) / tz + (cam.cy - (T)0.5);
  if (!finite_t(o.radius_f) || !finite_t(o.mu[0]) || !finite_t(o.mu[1])) return;
  const T rf = std::min(o.radius_f, (T)1073741824.0);
  o.radius = (int)rf;
  // 7. tile rect (clamp in floating point before the integer conversion)
  const T Gx = (T)((cam.width + 15) / 16), Gy = (T)((cam.height + 15) / 16);
  o.rect[0] = (int)std::min(Gx, std::max((T)0, std::floor((o.mu[0] - rf) / (T)16)));
  o.rect[1] = (int)std::min(Gy, std::max((T)0, std::floor((o.mu[1] - rf) / (T)16)));
  o.rect[2] = (int)std::min(Gx, std::max((T)0, std::floor(((o.mu[0] + rf) + (T)15) / (T)16)));
  o.rect[3] = (int)std::min(Gy, std::max((T)0, std::floor(((o.mu[1] + rf) + (T)15) / (T)16)));
  const int nx = o.rect[2] - o.rect[0], ny = o.rect[3] - o.rect[1];
  if (nx <= 0 || ny <= 0) return;
  o.tiles = (uint32_t)nx * (uint32_t)ny;
  // 8. colour: SH in the direction camera centre -> mean
  T cp[3];
  for (int k = 0; k < 3; ++k) cp[k] = -((W[k] * W[3] + W[4 + k] * W[7]) + W[8 + k] * W[11]);
  for (int k = 0; k < 3; ++k) o.dir[k] = p[k] - cp[k];
  o.dirlen = std::sqrt((o.dir[0] * o.dir[0] + o.dir[1] * o.dir[1]) + o.dir[2] * o.dir[2]);
  for (int k = 0; k < 3; ++k) o.dhat[k] = o.dir[k] / o.dirlen;
  sh_basis(o.dhat, sh_degree, o.basis);
  const int nb = (sh_degree + 1) * (sh_degree + 1);
  for (int ch = 0; ch < 3; ++ch) {
    T acc = o.basis[0] * sh[ch];
    for (int k = 1; k < nb; ++k) acc = acc + o.basis[k] * sh[3 * k + ch];
    acc = acc + (T)0.5;
    o.rgb_raw[ch] = acc;
    if (acc < (T)0) { o.clamped |= (uint8_t)(1u << ch); acc = (T)0; }
    o.rgb[ch] = acc;
  }
  if (o.clampx) o.clamped |= 8;
  if (o.clampy) o.clamped |= 16;
  o.visible = true;
}

template <class T>
Cam<T> make_cam(const double* cam, int width, int height) {
  Cam<T> c;
  c.fx = (T)cam[0]; c.fy = (T)cam[1]; c.cx = (T)cam[2]; c.cy = (T)cam[3];
  for (int k = 0; k < 12; ++k) c.W[k] = (T)cam[4 + k];
  c.near_plane = (T)cam[16];
  c.width = width; c.height = height;
  return c;
}

template <class T>
void project_index(int64_t i, int sh_degree, int sh_stored, const double* means, const double* scales,
                   const double* quats, const double* sh, const Cam<T>& cam, Proj<T>& o) {
  T p[3], s[3], q[4];
  for (int k = 0; k < 3; ++k) { p[k] = (T)means[3 * i + k]; s[k] = (T)scales[3 * i + k]; }
  for (int k = 0; k < 4; ++k) q[k] = (T)quats[4 * i + k];
  T c[48];
  const int nb = (sh_degree + 1) * (sh_degree + 1);
  for (int k = 0; k < nb * 3; ++k) c[k] = (T)sh[(size_t)i * sh_stored * 3 + k];
  project_one<T>(p, s, q, c, sh_degree, cam, o);
}

inline uint32_t float_bits(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }

}  // namespace

// ===================================================================================================
// C interface (plain pointers; all floating-point arrays are double; fp32 results are stored exactly
// in doubles so that callers can cast back to float32 and compare bit patterns).

extern "C" {

// Projection of every Gaussian (steps 1-8). mode 0: rule P-0 fp32; mode 1: fp64.
// cam = {fx, fy, cx, cy, w2c[12], near, bg[3]} (20 doubles).
int oracle_project(int mode, int64_t n, int sh_degree, int sh_stored, const double* means, const double* scales,
                   const double* quats, const double* opac, const double* sh, const double* cam, int width,
                   int height, double* depth, int32_t* radius, int32_t* rect, double* mean2d,
                   double* conic_opacity, double* rgb, uint8_t* clamped, uint32_t* tiles_touched) {
  if (sh_degree < 0 || sh_degree > 3 || sh_stored < (sh_degree + 1) * (sh_degree + 1)) return -1;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double d = 0, m0 = 0, m1 = 0, A = 0, B = 0, C = 0, r0 = 0, r1 = 0, r2 = 0;
    int rad = 0, rc[4] = {0, 0, 0, 0};
    uint8_t cl = 0;
    uint32_t tiles = 0;
    if (mode == 0) {
      Cam<float> c = make_cam<float>(cam, width, height);
      Proj<float> o;
      project_index<float>(i, sh_degree, sh_stored, means, scales, quats, sh, c, o);
      d = o.t[2];
      if (o.visible) {
        m0 = o.mu[0]; m1 = o.mu[1]; A = o.A; B = o.B; C = o.C; r0 = o.rgb[0]; r1 = o.rgb[1]; r2 = o.rgb[2];
        rad = o.radius; for (int k = 0; k < 4; ++k) rc[k] = o.rect[k];
        cl = o.clamped; tiles = o.tiles;
      }
    } else {
      Cam<double> c = make_cam<double>(cam, width, height);
      Proj<double> o;
      project_index<double>(i, sh_degree, sh_stored, means, scales, quats, sh, c, o);
      d = o.t[2];
      if (o.visible) {
        m0 = o.mu[0]; m1 = o.mu[1]; A = o.A; B = o.B; C = o.C; r0 = o.rgb[0]; r1 = o.rgb[1]; r2 = o.rgb[2];
        rad = o.radius; for (int k = 0; k < 4; ++k) rc[k] = o.rect[k];
        cl = o.clamped; tiles = o.tiles;
      }
    }
    depth[i] = d;
    radius[i] = rad;
    for (int k = 0; k < 4; ++k) rect[4 * i + k] = rc[k];
    mean2d[2 * i] = m0; mean2d[2 * i + 1] = m1;
    conic_opacity[4 * i] = A; conic_opacity[4 * i + 1] = B; conic_opacity[4 * i + 2] = C;
    conic_opacity[4 * i + 3] = tiles ? opac[i] : 0.0;
    rgb[3 * i] = r0; rgb[3 * i + 1] = r1; rgb[3 * i + 2] = r2;
    clamped[i] = cl;
    tiles_touched[i] = tiles;
  }
  return 0;
}

// Step 9: brute-force tile lists. Emission in index order, tiles row-major inside the rect, then
// std::stable_sort on the 64-bit key (tile << 32 | float_bits(depth)). Returns D; writes keys[D], vals[D]
// and ranges[ntiles][2] ((0,0) for empty tiles). Call with keys == NULL to get D only.
int64_t oracle_tile_lists(int64_t n, const double* depth, const int32_t* rect, const uint32_t* tiles_touched,
                          int grid_x, int ntiles, uint64_t* keys, uint32_t* vals, uint32_t* ranges) {
  int64_t D = 0;
  for (int64_t i = 0; i < n; ++i) D += tiles_touched[i];
  if (!keys) return D;
  std::vector<std::pair<uint64_t, uint32_t>> kv;
  kv.reserve((size_t)D);
  for (int64_t i = 0; i < n; ++i) {
    if (!tiles_touched[i]) continue;
    const uint32_t db = float_bits((float)depth[i]);
    for (int ty = rect[4 * i + 1]; ty < rect[4 * i + 3]; ++ty)
      for (int tx = rect[4 * i]; tx < rect[4 * i + 2]; ++tx) {
        const uint64_t tile = (uint64_t)ty * (uint64_t)grid_x + (uint64_t)tx;
        kv.emplace_back((tile << 32) | db, (uint32_t)i);
      }
  }
  std::stable_sort(kv.begin(), kv.end(),
                   [](const std::pair<uint64_t, uint32_t>& a, const std::pair<uint64_t, uint32_t>& b) { return a.first < b.first; });
  for (int t = 0; t < ntiles; ++t) ranges[2 * t] = ranges[2 * t + 1] = 0;
  for (int64_t k = 0; k < D; ++k) {
    keys[k] = kv[(size_t)k].first;
    vals[k] = kv[(size_t)k].second;
    const uint32_t tile = (uint32_t)(keys[k] >> 32);
    if (k == 0 || tile != (uint32_t)(keys[k - 1] >> 32)) ranges[2 * tile] = (uint32_t)k;
    ranges[2 * tile + 1] = (uint32_t)(k + 1);
  }
  return D;
}

}  // extern "C"

namespace {

// Global front-to-back order: visible Gaussians by (depth, index). Depths are positive, so ordering by
// value equals ordering by fp32 bit pattern in mode 0.
std::vector<int64_t> global_order(int64_t n, const double* depth, const uint32_t* tiles_touched) {
  std::vector<int64_t> ord;
  for (int64_t i = 0; i < n; ++i)
    if (tiles_touched[i]) ord.push_back(i);
  std::stable_sort(ord.begin(), ord.end(), [&](int64_t a, int64_t b) { return depth[a] < depth[b]; });
  return ord;
}

struct Contributor {
  int64_t g;
  double alpha, T, gauss, dx, dy;
  bool clamped;
};

// One pixel, one walk over the global list.
// Returns: out[CH], n_contrib, n_walked; optionally the contributor list for reverse-mode.
struct PixelResult {
  double Tfinal;
  uint32_t n_contrib, n_walked;
  uint8_t fragile;
  uint64_t examined, blended;
};

PixelResult composite_pixel(const std::vector<int64_t>& ord, int F, int CH, const double* depth, const int32_t* rect,
                            const double* mean2d, const double* conic_opacity, const double* rgb, const double* sem,
                            const double* unc, const double* bg, int px, int py, double fragile_rel, double* out,
                            std::vector<Contributor>* rec) {
  PixelResult r;
  r.Tfinal = 1.0; r.n_contrib = 0; r.n_walked = 0; r.fragile = 0; r.examined = 0; r.blended = 0;
  for (int c = 0; c < CH; ++c) out[c] = 0.0;
  const int tx = px / 16, ty = py / 16;
  const double alpha_min = 1.0 / 255.0, t_min = 1e-4, alpha_max = 0.99;
  double T = 1.0;
  uint32_t walked = 0;
  bool done = false;
  for (size_t k = 0; k < ord.size() && !done; ++k) {
    const int64_t g = ord[k];
    const int32_t* rc = rect + 4 * g;
    if (!(rc[0] <= tx && tx < rc[2] && rc[1] <= ty && ty < rc[3])) continue;
    ++walked;
    ++r.examined;
    const double dx = (double)px - mean2d[2 * g], dy = (double)py - mean2d[2 * g + 1];
    const double A = conic_opacity[4 * g], B = conic_opacity[4 * g + 1], C = conic_opacity[4 * g + 2], o = conic_opacity[4 * g + 3];
    const double power = -0.5 * (A * dx * dx + C * dy * dy) - B * dx * dy;
    if (std::fabs(power) < 1e-6) r.fragile |= 1;
    if (power > 0.0) continue;
    const double gauss = std::exp(power);
    const double raw = o * gauss;
    const double alpha = std::min(alpha_max, raw);
    if (std::fabs(alpha - alpha_min) < fragile_rel * alpha_min) r.fragile |= 1;
    if (std::fabs(raw - alpha_max) < fragile_rel * alpha_max) r.fragile |= 2;  // matters for gradients only
    if (alpha < alpha_min) continue;
    const double Tn = T * (1.0 - alpha);
    if (std::fabs(Tn - t_min) < fragile_rel * t_min) r.fragile |= 1;
    if (Tn < t_min) { done = true; break; }
    const double w = alpha * T;
    out[0] += w * rgb[3 * g]; out[1] += w * rgb[3 * g + 1]; out[2] += w * rgb[3 * g + 2];
    out[3] += w * depth[g];
    for (int f = 0; f < F; ++f) out[4 + f] += w * sem[(size_t)g * F + f];
    out[4 + F] += w * unc[g];
    if (rec) rec->push_back(Contributor{g, alpha, T, gauss, dx, dy, raw > alpha_max});
    T = Tn;
    r.n_contrib = walked;
    ++r.blended;
  }
  r.n_walked = walked;
  out[0] += T * bg[0]; out[1] += T * bg[1]; out[2] += T * bg[2];
  out[5 + F] = 1.0 - T;
  r.Tfinal = T;
  return r;
}

}  // namespace

extern "C" {

// Forward compositing of selected pixels. pix == NULL: all W*H pixels in row-major order (npix = W*H).
// pix[k] = py*W + px. out[npix][CH] layout: 0-2 rgb, 3 depth, 4..4+F-1 sem, 4+F unc, 5+F alpha=1-T, rest 0.
// counters[0] = examined pairs, [1] = blended pairs.
int oracle_composite_forward(int64_t n, int F, const double* depth, const int32_t* rect, const uint32_t* tiles_touched,
                             const double* mean2d, const double* conic_opacity, const double* rgb, const double* sem,
                             const double* unc, int width, int height, const double* bg, int64_t npix,
                             const int64_t* pix, double fragile_rel, double* out, uint32_t* n_contrib,
                             uint32_t* n_walked, uint8_t* fragile, uint64_t* counters) {
  const int CH = (3 + 1 + F + 1 + 1 + 3) / 4 * 4;
  const std::vector<int64_t> ord = global_order(n, depth, tiles_touched);
  uint64_t ex = 0, bl = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : ex, bl)
  for (int64_t k = 0; k < npix; ++k) {
    const int64_t p = pix ? pix[k] : k;
    const int px = (int)(p % width), py = (int)(p / width);
    (void)height;
    PixelResult r = composite_pixel(ord, F, CH, depth, rect, mean2d, conic_opacity, rgb, sem, unc, bg, px, py,
                                    fragile_rel, out + (size_t)k * CH, nullptr);
    if (n_contrib) n_contrib[k] = r.n_contrib;
    if (n_walked) n_walked[k] = r.n_walked;
    if (fragile) fragile[k] = r.fragile;
    ex += r.examined; bl += r.blended;
  }
  if (counters) { counters[0] = ex; counters[1] = bl; }
  return 0;
}

// Reverse-mode through the compositing of the selected pixels (SURVEY.md 8(c) "Backward").
// dL_dpix[npix][CH]: only rgb (0-2), sem (4..4+F-1) and unc (4+F) slots are read.
// flags bit1: semantic + uncertainty upstream gradients also flow into alpha (geometry); default (0) they reach
// only dsem / dunc (reading C-14 of PAPER.md:182).
// Outputs are ACCUMULATED into (caller zeroes): dopac[n], dconic[n][3], dmean2d[n][2], drgb[n][3], dsem[n][F], dunc[n].
// flags bit2 (reading C-17b: upstream gradients for the depth and alpha images): the depth slot (3)
// and the alpha slot (5+F) of dL_dpix are read too. depth_out = sum_k w_k z_k is one more blended channel (value z_k = the
// view-space depth, which reaches the geometry: dL/dalpha gets G_3 (T z - S_3/(1-alpha)) and ddepth[g] += w G_3 is the
// gradient with respect to z_g); alpha_out = 1 - T_final = 1 - prod_j (1 - alpha_j), so d alpha_out / d alpha_k =
// T_final / (1 - alpha_k): the same form as a background of -1 on a channel whose values are all 0.
// ddepth [n] (may be NULL when bit2 is clear): accumulated into.
int oracle_composite_backward(int64_t n, int F, const double* depth, const int32_t* rect, const uint32_t* tiles_touched,
                              const double* mean2d, const double* conic_opacity, const double* rgb, const double* sem,
                              const double* unc, int width, int height, const double* bg, int64_t npix,
                              const int64_t* pix, const double* dL_dpix, int flags, double* dopac, double* dconic,
                              double* dmean2d, double* drgb, double* dsem, double* dunc, double* ddepth) {
  const int CH = (3 + 1 + F + 1 + 1 + 3) / 4 * 4;
  const bool couple = (flags & 2) != 0;
  const bool geo = (flags & 4) != 0;   // depth and alpha upstream gradients
  if (geo && !ddepth) return -1;
  const std::vector<int64_t> ord = global_order(n, depth, tiles_touched);
  (void)height;
#pragma omp parallel
  {
    std::vector<Contributor> rec;
    std::vector<double> out((size_t)CH), S((size_t)CH);
#pragma omp for schedule(dynamic, 16)
    for (int64_t k = 0; k < npix; ++k) {
      const int64_t p = pix ? pix[k] : k;
      const int px = (int)(p % width), py = (int)(p / width);
      rec.clear();
      PixelResult r = composite_pixel(ord, F, CH, depth, rect, mean2d, conic_opacity, rgb, sem, unc, bg, px, py, 0.0,
                                      out.data(), &rec);
      const double* G = dL_dpix + (size_t)k * CH;
      // suffix sums S_ch = sum_{j>k} w_j v_j,ch + T_final * bg_ch
      for (int c = 0; c < CH; ++c) S[c] = 0.0;
      S[0] = r.Tfinal * bg[0]; S[1] = r.Tfinal * bg[1]; S[2] = r.Tfinal * bg[2];
      if (geo) S[5 + F] = -r.Tfinal;   // alpha_out - 1 = -T_final: "background" -1, values 0
      for (size_t m = rec.size(); m-- > 0;) {
        const Contributor& q = rec[m];
        const int64_t g = q.g;
        const double w = q.alpha * q.T;
        double dLda = 0.0;
        const double inv1ma = 1.0 / (1.0 - q.alpha);
        for (int c = 0; c < 3; ++c) {
          const double v = rgb[3 * g + c];
#pragma omp atomic
          drgb[3 * g + c] += w * G[c];
          dLda += G[c] * (q.T * v - S[c] * inv1ma);
          S[c] += w * v;
        }
        for (int f = 0; f < F; ++f) {
          const double v = sem[(size_t)g * F + f];
#pragma omp atomic
          dsem[(size_t)g * F + f] += w * G[4 + f];
          if (couple) dLda += G[4 + f] * (q.T * v - S[4 + f] * inv1ma);
          S[4 + f] += w * v;
        }
        {
          const double v = unc[g];
#pragma omp atomic
          dunc[g] += w * G[4 + F];
          if (couple) dLda += G[4 + F] * (q.T * v - S[4 + F] * inv1ma);
          S[4 + F] += w * v;
        }
        if (geo) {
          const double v = depth[g];
#pragma omp atomic
          ddepth[g] += w * G[3];
          dLda += G[3] * (q.T * v - S[3] * inv1ma);
          S[3] += w * v;
          dLda += G[5 + F] * (-S[5 + F] * inv1ma);   // the alpha image: every value is 0, only the "background" term
        }
        if (q.clamped) continue;  // alpha saturated at 0.99: zero derivative (reading C-15)
        const double A = conic_opacity[4 * g], B = conic_opacity[4 * g + 1], C = conic_opacity[4 * g + 2], o = conic_opacity[4 * g + 3];
        const double dpow = o * q.gauss * dLda;
#pragma omp atomic
        dopac[g] += q.gauss * dLda;
#pragma omp atomic
        dmean2d[2 * g] += dpow * (A * q.dx + B * q.dy);
#pragma omp atomic
        dmean2d[2 * g + 1] += dpow * (C * q.dy + B * q.dx);
#pragma omp atomic
        dconic[3 * g] += dpow * (-0.5 * q.dx * q.dx);
#pragma omp atomic
        dconic[3 * g + 1] += dpow * (-q.dx * q.dy);
#pragma omp atomic
        dconic[3 * g + 2] += dpow * (-0.5 * q.dy * q.dy);
      }
    }
  }
  return 0;
}

// Conditioning of the sums oracle_composite_backward forms (reading G-4 of SURVEY.md 8(c) / DESIGN.md: an fp32 accumulation in
// any order can only be held to a multiple of 2^-24 sum|term|). NOT part of the method and no gradient: the same walk over the
// same contributors, but every product the gradient expands into is taken by absolute value before it is added, down to the
// single products (per pixel and per channel: dL/dalpha_k is itself a sum over channels of G_ch T_k v_k,ch, of
// - G_ch w_j v_j,ch / (1 - alpha_k) for every later contributor j, and of - G_ch T_final bg_ch / (1 - alpha_k); the two terms
// of A dx + B dy count apart).
// abs_sums [n][10 + F (+ 1 with flags bit2)] (caller zeroes), in the order dopac, dconic[3], dmean2d[2], drgb[3], dsem[F],
// dunc (, ddepth). Pinned in tests/test_oracle_conditioning.py (>= |gradient|; equality for one-signed sums; an explicit numpy
// expansion on a small scene).
int oracle_composite_backward_abs(int64_t n, int F, const double* depth, const int32_t* rect, const uint32_t* tiles_touched,
                                  const double* mean2d, const double* conic_opacity, const double* rgb, const double* sem,
                                  const double* unc, int width, int height, const double* bg, int64_t npix,
                                  const int64_t* pix, const double* dL_dpix, int flags, double* abs_sums) {
  const int CH = (3 + 1 + F + 1 + 1 + 3) / 4 * 4;
  const bool couple = (flags & 2) != 0;
  const bool geo = (flags & 4) != 0;
  if (!abs_sums) return -1;
  const size_t NS = (size_t)(10 + F + (geo ? 1 : 0));
  const std::vector<int64_t> ord = global_order(n, depth, tiles_touched);
  (void)height;
#pragma omp parallel
  {
    std::vector<Contributor> rec;
    std::vector<double> out((size_t)CH), Sabs((size_t)CH);
#pragma omp for schedule(dynamic, 16)
    for (int64_t k = 0; k < npix; ++k) {
      const int64_t p = pix ? pix[k] : k;
      const int px = (int)(p % width), py = (int)(p / width);
      rec.clear();
      PixelResult r = composite_pixel(ord, F, CH, depth, rect, mean2d, conic_opacity, rgb, sem, unc, bg, px, py, 0.0,
                                      out.data(), &rec);
      const double* G = dL_dpix + (size_t)k * CH;
      // Sabs_ch = sum_{j>k} w_j |v_j,ch| + T_final |bg_ch|: the suffix sums of the gradient with every product made positive
      for (int c = 0; c < CH; ++c) Sabs[c] = 0.0;
      for (int c = 0; c < 3; ++c) Sabs[c] = std::fabs(r.Tfinal * bg[c]);
      if (geo) Sabs[5 + F] = r.Tfinal;
      auto add = [&](int64_t g, size_t slot, double term) {
#pragma omp atomic
        abs_sums[(size_t)g * NS + slot] += std::fabs(term);
      };
      for (size_t m = rec.size(); m-- > 0;) {
        const Contributor& q = rec[m];
        const int64_t g = q.g;
        const double w = q.alpha * q.T;
        const double inv1ma = 1.0 / (1.0 - q.alpha);
        double adLda = 0.0;   // sum of |G_ch| (T |v| + Sabs/(1-alpha)): dL/dalpha with every product made positive
        for (int c = 0; c < 3; ++c) {
          const double v = std::fabs(rgb[3 * g + c]);
          add(g, 6 + c, w * G[c]);
          adLda += std::fabs(G[c]) * (q.T * v + Sabs[c] * inv1ma);
          Sabs[c] += w * v;
        }
        for (int f = 0; f < F; ++f) {
          const double v = std::fabs(sem[(size_t)g * F + f]);
          add(g, 9 + f, w * G[4 + f]);
          if (couple) adLda += std::fabs(G[4 + f]) * (q.T * v + Sabs[4 + f] * inv1ma);
          Sabs[4 + f] += w * v;
        }
        {
          const double v = std::fabs(unc[g]);
          add(g, 9 + F, w * G[4 + F]);
          if (couple) adLda += std::fabs(G[4 + F]) * (q.T * v + Sabs[4 + F] * inv1ma);
          Sabs[4 + F] += w * v;
        }
        if (geo) {
          const double v = std::fabs(depth[g]);
          add(g, 10 + F, w * G[3]);
          adLda += std::fabs(G[3]) * (q.T * v + Sabs[3] * inv1ma);
          Sabs[3] += w * v;
          adLda += std::fabs(G[5 + F]) * (Sabs[5 + F] * inv1ma);
        }
        if (q.clamped) continue;
        const double A = conic_opacity[4 * g], B = conic_opacity[4 * g + 1], C = conic_opacity[4 * g + 2], o = conic_opacity[4 * g + 3];
        const double ap = std::fabs(o * q.gauss) * adLda;
        add(g, 0, q.gauss * adLda);
        add(g, 1, ap * (0.5 * q.dx * q.dx));
        add(g, 2, ap * (q.dx * q.dy));
        add(g, 3, ap * (0.5 * q.dy * q.dy));
        add(g, 4, ap * (std::fabs(A * q.dx) + std::fabs(B * q.dy)));
        add(g, 5, ap * (std::fabs(C * q.dy) + std::fabs(B * q.dx)));
      }
    }
  }
  return 0;
}

}  // extern "C"

// ===================================================================================================
// Per-Gaussian projection backward: derivative formulas evaluated in
// fp64 on the intermediates of the forward projection (mode 0: the fp32 intermediates, widened).

namespace {

template <class T>
Proj<double> widen(const Proj<T>& s) {
  Proj<double> d;
  d.visible = s.visible;
  for (int k = 0; k < 3; ++k) { d.t[k] = s.t[k]; d.dir[k] = s.dir[k]; d.dhat[k] = s.dhat[k]; d.rgb[k] = s.rgb[k]; d.rgb_raw[k] = s.rgb_raw[k]; }
  for (int k = 0; k < 9; ++k) { d.R[k] = s.R[k]; d.M[k] = s.M[k]; }
  for (int k = 0; k < 6; ++k) { d.Sig[k] = s.Sig[k]; d.Tm[k] = s.Tm[k]; }
  d.xt = s.xt; d.yt = s.yt; d.clampx = s.clampx; d.clampy = s.clampy;
  d.J00 = s.J00; d.J02 = s.J02; d.J11 = s.J11; d.J12 = s.J12;
  d.a = s.a; d.b = s.b; d.c = s.c; d.det = s.det; d.A = s.A; d.B = s.B; d.C = s.C;
  d.mu[0] = s.mu[0]; d.mu[1] = s.mu[1]; d.radius_f = s.radius_f; d.radius = s.radius;
  for (int k = 0; k < 4; ++k) d.rect[k] = s.rect[k];
  d.tiles = s.tiles; d.dirlen = s.dirlen;
  for (int k = 0; k < 16; ++k) d.basis[k] = s.basis[k];
  d.clamped = s.clamped;
  return d;
}

// o: forward intermediates; q, s: quaternion and scale; sh: [stored,3] coefficients; cam in double.
// Upstream: gconic[3] (dL/dA, dL/dB, dL/dC), gmu[2], grgb[3] (w.r.t. the clamped colour), gdepth (w.r.t. the view-space
// depth t_z that the depth image blends; 0 unless the depth image has an upstream gradient).
void project_backward_one(const Proj<double>& o, const double q[4], const double s[3], const double* sh, int sh_degree,
                          const Cam<double>& cam, const double gconic[3], const double gmu[2], const double grgb[3],
                          double gdepth, double dmean[3], double dscale[3], double dquat[4], double* dsh /*[stored,3]*/) {
  const double* W = cam.W;
  // conic -> dilated covariance: Q = [[A,B],[B,C]], dQ = [[gA, gB/2],[gB/2, gC]], dCov = -Q dQ Q
  const double Q00 = o.A, Q01 = o.B, Q11 = o.C;
  const double D00 = gconic[0], D01 = 0.5 * gconic[1], D11 = gconic[2];
  // P = Q dQ
  const double P00 = Q00 * D00 + Q01 * D01, P01 = Q00 * D01 + Q01 * D11;
  const double P10 = Q01 * D00 + Q11 * D01, P11 = Q01 * D01 + Q11 * D11;
  // G = -(P Q)
  const double G00 = -(P00 * Q00 + P01 * Q01), G01 = -(P00 * Q01 + P01 * Q11);
  const double G11 = -(P10 * Q01 + P11 * Q11);
  const double Gp[2][2] = {{G00, G01}, {G01, G11}};  // full symmetric gradient of the 2x2 covariance
  const double Tm[2][3] = {{o.Tm[0], o.Tm[1], o.Tm[2]}, {o.Tm[3], o.Tm[4], o.Tm[5]}};
  const double Sg[3][3] = {{o.Sig[0], o.Sig[1], o.Sig[2]}, {o.Sig[1], o.Sig[3], o.Sig[4]}, {o.Sig[2], o.Sig[4], o.Sig[5]}};
  // dSigma = T^T G' T   (3x3)
  double GT[2][3];
  for (int i = 0; i < 2; ++i)
    for (int k = 0; k < 3; ++k) GT[i][k] = Gp[i][0] * Tm[0][k] + Gp[i][1] * Tm[1][k];
  double dSig[3][3];
  for (int i = 0; i < 3; ++i)
    for (int k = 0; k < 3; ++k) dSig[i][k] = Tm[0][i] * GT[0][k] + Tm[1][i] * GT[1][k];
  // dT = 2 G' T Sigma   (2x3)
  double dT[2][3];
  for (int i = 0; i < 2; ++i)
    for (int k = 0; k < 3; ++k) dT[i][k] = 2.0 * (GT[i][0] * Sg[0][k] + GT[i][1] * Sg[1][k] + GT[i][2] * Sg[2][k]);
  // dJ = dT R_wc^T ; only the four structurally non-zero entries of J matter
  auto dJ = [&](int i, int j) { return dT[i][0] * W[4 * j] + dT[i][1] * W[4 * j + 1] + dT[i][2] * W[4 * j + 2]; };
  const double dJ00 = dJ(0, 0), dJ02 = dJ(0, 2), dJ11 = dJ(1, 1), dJ12 = dJ(1, 2);
  const double tx = o.t[0], ty = o.t[1], tz = o.t[2];
  const double fx = cam.fx, fy = cam.fy;
  const double tz2 = tz * tz;
  double dt[3] = {0, 0, 0};
  // J02 = -fx*xt/tz^2 with xt = tx (unclamped) or +-limx*tz (clamped)
  if (!o.clampx) { dt[0] += dJ02 * (-fx / tz2); dt[2] += dJ02 * (2.0 * fx * tx / (tz2 * tz)); }
  else           { dt[2] += dJ02 * (-o.J02 / tz); }
  if (!o.clampy) { dt[1] += dJ12 * (-fy / tz2); dt[2] += dJ12 * (2.0 * fy * ty / (tz2 * tz)); }
  else           { dt[2] += dJ12 * (-o.J12 / tz); }
  dt[2] += dJ00 * (-fx / tz2) + dJ11 * (-fy / tz2);
  // mean2D = (fx tx/tz + cx - .5, fy ty/tz + cy - .5)
  dt[0] += gmu[0] * (fx / tz);
  dt[1] += gmu[1] * (fy / tz);
  dt[2] += gmu[0] * (-fx * tx / tz2) + gmu[1] * (-fy * ty / tz2);
  dt[2] += gdepth;   // depth = t_z (step 1)
  for (int k = 0; k < 3; ++k) dmean[k] = W[k] * dt[0] + W[4 + k] * dt[1] + W[8 + k] * dt[2];
  // Sigma = M M^T -> dM = 2 dSigma M ; M = R diag(s)
  double dM[3][3];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j)
      dM[i][j] = 2.0 * (dSig[i][0] * o.M[j] + dSig[i][1] * o.M[3 + j] + dSig[i][2] * o.M[6 + j]);
  double dR[3][3];
  for (int j = 0; j < 3; ++j) {
    dscale[j] = o.R[j] * dM[0][j] + o.R[3 + j] * dM[1][j] + o.R[6 + j] * dM[2][j];
    for (int i = 0; i < 3; ++i) dR[i][j] = dM[i][j] * s[j];
  }
  const double w = q[0], x = q[1], y = q[2], z = q[3];
  dquat[0] = 2.0 * (-z * dR[0][1] + y * dR[0][2] + z * dR[1][0] - x * dR[1][2] - y * dR[2][0] + x * dR[2][1]);
  dquat[1] = 2.0 * (y * dR[0][1] + z * dR[0][2] + y * dR[1][0] - 2.0 * x * dR[1][1] - w * dR[1][2] + z * dR[2][0] + w * dR[2][1] - 2.0 * x * dR[2][2]);
  dquat[2] = 2.0 * (-2.0 * y * dR[0][0] + x * dR[0][1] + w * dR[0][2] + x * dR[1][0] + z * dR[1][2] - w * dR[2][0] + z * dR[2][1] - 2.0 * y * dR[2][2]);
  dquat[3] = 2.0 * (-2.0 * z * dR[0][0] - w * dR[0][1] + x * dR[0][2] + w * dR[1][0] - 2.0 * z * dR[1][1] + y * dR[1][2] + x * dR[2][0] + y * dR[2][1]);
  // colour: rgb = max(0, 0.5 + sum_k Y_k(dhat) c_k)
  const int nb = (sh_degree + 1) * (sh_degree + 1);
  double g[3];
  for (int ch = 0; ch < 3; ++ch) g[ch] = (o.clamped & (1u << ch)) ? 0.0 : grgb[ch];
  double bg[16][3];
  sh_basis_grad<double>(o.dhat, sh_degree, bg);
  double ddhat[3] = {0, 0, 0};
  for (int k = 0; k < nb; ++k) {
    double cg = 0.0;
    for (int ch = 0; ch < 3; ++ch) { dsh[3 * k + ch] = o.basis[k] * g[ch]; cg += sh[3 * k + ch] * g[ch]; }
    for (int a = 0; a < 3; ++a) ddhat[a] += bg[k][a] * cg;
  }
  const double dot = o.dhat[0] * ddhat[0] + o.dhat[1] * ddhat[1] + o.dhat[2] * ddhat[2];
  for (int a = 0; a < 3; ++a) dmean[a] += (ddhat[a] - o.dhat[a] * dot) / o.dirlen;
}

}  // namespace

extern "C" {

// Upstream per-Gaussian gradients (from oracle_composite_backward) -> gradients of the 3D parameters.
// Outputs (overwritten): dmeans[n][3], dscales[n][3], dquats[n][4], dsh[n][sh_stored][3]. Culled Gaussians get 0.
int oracle_project_backward(int mode, int64_t n, int sh_degree, int sh_stored, const double* means, const double* scales,
                            const double* quats, const double* sh, const double* cam, int width, int height,
                            const double* gconic, const double* gmean2d, const double* grgb, double* dmeans,
                            double* dscales, double* dquats, double* dsh, const double* gdepth /* [n] or NULL */) {
  const Cam<double> camd = make_cam<double>(cam, width, height);
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    for (int k = 0; k < 3; ++k) dmeans[3 * i + k] = dscales[3 * i + k] = 0.0;
    for (int k = 0; k < 4; ++k) dquats[4 * i + k] = 0.0;
    for (int k = 0; k < sh_stored * 3; ++k) dsh[(size_t)i * sh_stored * 3 + k] = 0.0;
    Proj<double> o;
    if (mode == 0) {
      Cam<float> c = make_cam<float>(cam, width, height);
      Proj<float> of;
      project_index<float>(i, sh_degree, sh_stored, means, scales, quats, sh, c, of);
      if (!of.visible) continue;
      o = widen(of);
    } else {
      project_index<double>(i, sh_degree, sh_stored, means, scales, quats, sh, camd, o);
      if (!o.visible) continue;
    }
    project_backward_one(o, quats + 4 * i, scales + 3 * i, sh + (size_t)i * sh_stored * 3, sh_degree, camd,
                         gconic + 3 * i, gmean2d + 2 * i, grgb + 3 * i, gdepth ? gdepth[i] : 0.0, dmeans + 3 * i, dscales + 3 * i, dquats + 4 * i,
                         dsh + (size_t)i * sh_stored * 3);
  }
  return 0;
}

// SH basis values for a unit direction (exposed for the Gram-matrix quadrature pin).
void oracle_sh_basis(const double* dir, int degree, double* out16) {
  for (int k = 0; k < 16; ++k) out16[k] = 0.0;
  sh_basis<double>(dir, degree, out16);
}

// ---------------------------------------------------------------------------------------------------
// Relevancy of a given feature map ("the relevance map of F", read as the plain cosine, C-21; SURVEY.md 8(b)
// input_is_probs = 0): rel[p][q] = <F_p[0:d_clip], query_q> / (|F_p[0:d_clip]| |query_q|), F [P][d]. A zero row gives 0.
int oracle_relevancy_map(int64_t P, int d, int d_clip, const double* F, const double* queries, int Q, double* rel) {
  for (int64_t p = 0; p < P; ++p) {
    double nf = 0.0;
    for (int j = 0; j < d_clip; ++j) nf += F[(size_t)p * d + j] * F[(size_t)p * d + j];
    for (int qi = 0; qi < Q; ++qi) {
      double dot = 0.0, nq = 0.0;
      for (int j = 0; j < d_clip; ++j) {
        dot += F[(size_t)p * d + j] * queries[(size_t)qi * d_clip + j];
        nq += queries[(size_t)qi * d_clip + j] * queries[(size_t)qi * d_clip + j];
      }
      rel[(size_t)p * Q + qi] = (nf > 0.0 && nq > 0.0) ? dot / (std::sqrt(nf) * std::sqrt(nq)) : 0.0;
    }
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------------
// Decode (Eq. 21-22, Table 3; relevancy PAPER.md:360 read as plain cosine, C-21).
// x[P][dims[0]]; layer l: W_l [dims[l+1]][dims[l]] row-major, b_l [dims[l+1]] (NULL = none); ReLU between
// layers, none after the last; probs = softmax(logits); decoded = probs^T * codebook [K][d];
// rel[q] = <decoded[0:d_clip], query_q> / (|decoded[0:d_clip]| |query_q|). Any output pointer may be NULL.
int oracle_decode(int64_t P, int n_layers, const int32_t* dims, const double* x, const double* const* W,
                  const double* const* b, const double* codebook, int d, int d_clip, const double* queries, int Q,
                  double* probs, double* decoded, double* rel) {
  const int K = dims[n_layers];
#pragma omp parallel
  {
    std::vector<double> h0, h1, dec((size_t)d);
#pragma omp for schedule(static)
    for (int64_t p = 0; p < P; ++p) {
      h0.assign(x + (size_t)p * dims[0], x + (size_t)(p + 1) * dims[0]);
      for (int l = 0; l < n_layers; ++l) {
        const int in = dims[l], out = dims[l + 1];
        h1.assign((size_t)out, 0.0);
        for (int oi = 0; oi < out; ++oi) {
          double acc = (b && b[l]) ? b[l][oi] : 0.0;
          for (int ii = 0; ii < in; ++ii) acc += W[l][(size_t)oi * in + ii] * h0[ii];
          if (l + 1 < n_layers && acc < 0.0) acc = 0.0;
          h1[oi] = acc;
        }
        h0.swap(h1);
      }
      double mx = h0[0];
      for (int k = 1; k < K; ++k) mx = std::max(mx, h0[k]);
      double sum = 0.0;
      for (int k = 0; k < K; ++k) { h0[k] = std::exp(h0[k] - mx); sum += h0[k]; }
      for (int k = 0; k < K; ++k) h0[k] /= sum;
      if (probs) for (int k = 0; k < K; ++k) probs[(size_t)p * K + k] = h0[k];
      if (decoded || rel) {
        for (int j = 0; j < d; ++j) {
          double acc = 0.0;
          for (int k = 0; k < K; ++k) acc += h0[k] * codebook[(size_t)k * d + j];
          dec[j] = acc;
        }
        if (decoded) for (int j = 0; j < d; ++j) decoded[(size_t)p * d + j] = dec[j];
        if (rel) {
          double nf = 0.0;
          for (int j = 0; j < d_clip; ++j) nf += dec[j] * dec[j];
          nf = std::sqrt(nf);
          for (int qi = 0; qi < Q; ++qi) {
            double dot = 0.0, nq = 0.0;
            for (int j = 0; j < d_clip; ++j) { dot += dec[j] * queries[(size_t)qi * d_clip + j]; nq += queries[(size_t)qi * d_clip + j] * queries[(size_t)qi * d_clip + j]; }
            rel[(size_t)p * Q + qi] = dot / (nf * std::sqrt(nq));
          }
        }
      }
    }
  }
  return 0;
}

// Semantic loss head (Eq. 8-12), forward and reverse mode, all fp64:
//   M^ = softmax(D_MLP(R_s)) (Eq. 8);  L_CE = sum_p CE(M^_p, M_p) (1 - R_u,p) / P (Eq. 10);  L_u = sum_p R_u,p / P (Eq. 11);
//   L_s = lambda_ce L_CE + lambda_u L_u (Eq. 12).  CE(M^_p, m) = -log M^_p[m] (reading: natural logarithm, mean over
//   H x W as Eq. 10 writes it). D_MLP as in oracle_decode: ReLU between layers, none after the last.
// x [P][dims[0]] = rendered compact feature R_s, u [P] = rendered uncertainty R_u, index [P] in [0, K).
// Outputs: loss[0] = L_CE, loss[1] = L_u, loss[2] = L_s; dx [P][dims[0]] = dL_s/dR_s; du [P] = dL_s/dR_u;
// dW[l] [dims[l+1]][dims[l]], db[l] [dims[l+1]] = dL_s/d(weights) (db[l] may be NULL). One pixel at a time, plain loops.
int oracle_semantic_loss(int64_t P, int n_layers, const int32_t* dims, const double* x, const double* u,
                         const int32_t* index, const double* const* W, const double* const* b, double lambda_ce,
                         double lambda_u, double* loss, double* dx, double* du, double* const* dW, double* const* db) {
  if (n_layers < 1 || n_layers > 3) return -1;
  const int K = dims[n_layers];
  double l_ce = 0.0, l_u = 0.0;
  std::vector<std::vector<double>> act(n_layers + 1), pre(n_layers + 1), g(n_layers + 1);
  for (int64_t p = 0; p < P; ++p) {
    if (index[p] < 0 || index[p] >= K) return -2;
    act[0].assign(x + (size_t)p * dims[0], x + (size_t)(p + 1) * dims[0]);
    for (int l = 0; l < n_layers; ++l) {
      const int in = dims[l], out = dims[l + 1];
      pre[l + 1].assign((size_t)out, 0.0);
      act[l + 1].assign((size_t)out, 0.0);
      for (int o = 0; o < out; ++o) {
        double a = (b && b[l]) ? b[l][o] : 0.0;
        for (int i = 0; i < in; ++i) a += W[l][(size_t)o * in + i] * act[l][i];
        pre[l + 1][o] = a;
        act[l + 1][o] = (l + 1 < n_layers && a < 0.0) ? 0.0 : a;
      }
    }
    const std::vector<double>& z = act[n_layers];
    double mx = z[0];
    for (int k = 1; k < K; ++k) mx = std::max(mx, z[k]);
    double sum = 0.0;
    for (int k = 0; k < K; ++k) sum += std::exp(z[k] - mx);
    const double ce = (mx + std::log(sum)) - z[index[p]];            // -log softmax(z)[m]
    l_ce += ce * (1.0 - u[p]);
    l_u += u[p];
    // reverse mode
    du[p] = (-lambda_ce * ce + lambda_u) / (double)P;
    const double coef = lambda_ce * (1.0 - u[p]) / (double)P;
    g[n_layers].assign((size_t)K, 0.0);
    for (int k = 0; k < K; ++k) g[n_layers][k] = coef * (std::exp(z[k] - mx) / sum - (k == index[p] ? 1.0 : 0.0));
    for (int l = n_layers - 1; l >= 0; --l) {
      const int in = dims[l], out = dims[l + 1];
      if (l + 1 < n_layers)
        for (int o = 0; o < out; ++o) if (!(pre[l + 1][o] > 0.0)) g[l + 1][o] = 0.0;   // ReLU: zero gradient at pre <= 0
      g[l].assign((size_t)in, 0.0);
      for (int o = 0; o < out; ++o) {
        const double go = g[l + 1][o];
        if (db && db[l]) db[l][o] += go;
        for (int i = 0; i < in; ++i) {
          dW[l][(size_t)o * in + i] += go * act[l][i];
          g[l][i] += W[l][(size_t)o * in + i] * go;
        }
      }
    }
    for (int i = 0; i < dims[0]; ++i) dx[(size_t)p * dims[0] + i] = g[0][i];
  }
  loss[0] = l_ce / (double)P;
  loss[1] = l_u / (double)P;
  loss[2] = lambda_ce * loss[0] + lambda_u * loss[1];
  return 0;
}

}  // extern "C"

// ===================================================================================================
// Training-step plumbing named at PAPER.md:182: "utilizing the Adam optimizer [25], with a
// learning rate set to 0.001 and betas equal to (0.9, 0.999)" and "adaptive density control of 3D Gaussians" following
// [17], which needs the accumulated screen-space positional gradient per Gaussian.
extern "C" {

// One Adam step (Kingma & Ba, Algorithm 1, with bias correction), fp64, in place, t = 1-based step count:
//   m <- b1 m + (1-b1) g;  v <- b2 v + (1-b2) g^2;  p <- p - lr (m / (1-b1^t)) / (sqrt(v / (1-b2^t)) + eps).
// eps is an argument (the paper gives lr and betas only; reading C-26: eps = 1e-8, the default of [25]).
int oracle_adam_step(int64_t count, double* p, const double* g, double* m, double* v, double lr, double beta1,
                     double beta2, double eps, int step) {
  if (step < 1) return -1;
  const double c1 = 1.0 - std::pow(beta1, (double)step), c2 = 1.0 - std::pow(beta2, (double)step);
  for (int64_t i = 0; i < count; ++i) {
    m[i] = beta1 * m[i] + (1.0 - beta1) * g[i];
    v[i] = beta2 * v[i] + (1.0 - beta2) * g[i] * g[i];
    const double mhat = m[i] / c1, vhat = v[i] / c2;
    p[i] = p[i] - lr * mhat / (std::sqrt(vhat) + eps);
  }
  return 0;
}

// Density-control statistics of one view (reading C-27 of "adaptive density control" following [17]):
// for every Gaussian visible in the view (radius > 0): grad_accum += |dL/dmean2d|_2 (pixels, reading C-16), denom += 1,
// max_radius = max(max_radius, radius). Invisible Gaussians are left untouched.
int oracle_density_stats(int64_t n, const double* dmean2d, const int32_t* radius, double* grad_accum, uint32_t* denom,
                         int32_t* max_radius) {
  for (int64_t i = 0; i < n; ++i) {
    if (radius[i] <= 0) continue;
    grad_accum[i] += std::sqrt(dmean2d[2 * i] * dmean2d[2 * i] + dmean2d[2 * i + 1] * dmean2d[2 * i + 1]);
    denom[i] += 1u;
    max_radius[i] = std::max(max_radius[i], radius[i]);
  }
  return 0;
}

}  // extern "C"

// ===================================================================================================
// LERF-style relevancy (optional). PAPER.md:360 only says the relevancy map is computed "in
// accordance with LERF [18]"; the formula is NOT in this paper and [18] is not in the container, so BY THE PAPER this
// function is "parity unpinned" (reading C-21b). It restates the published LERF score: with cos[p][j] the cosine
// of pixel p's decoded CLIP feature against positive query j (columns 0..n_pos-1 of the cosine map of oracle_decode) and
// against canonical negative phrase i (columns n_pos..Q-1),
//   out[p][j] = min_i  exp(tau cos[p][j]) / (exp(tau cos[p][j]) + exp(tau cos[p][n_pos + i]))
// i.e. the first entry of a two-way softmax at temperature 1/tau, minimised over the negatives.
extern "C" {
int oracle_relevancy_lerf(int64_t P, int Q, int n_pos, double tau, const double* cosines, double* out) {
  if (n_pos < 1 || n_pos >= Q) return -1;
  for (int64_t p = 0; p < P; ++p)
    for (int j = 0; j < n_pos; ++j) {
      double best = 2.0;
      for (int i = n_pos; i < Q; ++i) {
        const double a = std::exp(tau * cosines[(size_t)p * Q + j]), b = std::exp(tau * cosines[(size_t)p * Q + i]);
        best = std::min(best, a / (a + b));
      }
      out[(size_t)p * n_pos + j] = best;
    }
  return 0;
}
}  // extern "C"

// ===================================================================================================
// Quantisation search and codebook losses (SURVEY.md 8(f) item 2; PAPER.md:76-108 Eq. 3-7, :310-329 Eq. 16-20).
extern "C" {

// F [P][d] hybrid features (first d_clip dims = CLIP part, the rest = DINO part, Eq. 2), S [N][d] discrete feature space.
//   D(F, f_i) = cos<F^CLIP, f_i^CLIP> + lambda_dino cos<F^DINO, f_i^DINO>          (Eq. 4)
//   m_p = argmax_i D(F_p, f_i)  (Eq. 16; ties: the lowest index, reading C-28)     -> index [P]
//   r = sum_p onehot(m_p) / P (Eq. 17);  p = sum_p softmax_i(D(F_p, f_i)) / P (Eq. 18-19);  L_lb = sum_i r_i p_i (Eq. 20)
//   L_cos = mean_p [ (1 - cos<F_p^CLIP, f_m^CLIP>) + lambda_dino (1 - cos<F_p^DINO, f_m^DINO>) ]   (Eq. 5, averaged over
//   the quantised features: reading C-29);  L_q = lambda_cos L_cos + lambda_lb L_lb  (Eq. 7).
// Outputs (any may be NULL): index [P], gap [P] = D(best) - D(second best) (test infrastructure: near-tie flag),
// r [N], p [N], loss [3] = L_cos, L_lb, L_q, scores [P][N] = D.
int oracle_quantize(int64_t P, int N, int d, int d_clip, const double* F, const double* S, double lambda_dino,
                    double lambda_cos, double lambda_lb, int32_t* index, double* gap, double* r, double* p, double* loss,
                    double* scores) {
  if (N < 1 || d_clip < 1 || d_clip >= d) return -1;
  std::vector<double> nc((size_t)N), nd((size_t)N), rr((size_t)N, 0.0), pp((size_t)N, 0.0), D((size_t)N);
  for (int i = 0; i < N; ++i) {
    double a = 0.0, b = 0.0;
    for (int j = 0; j < d_clip; ++j) a += S[(size_t)i * d + j] * S[(size_t)i * d + j];
    for (int j = d_clip; j < d; ++j) b += S[(size_t)i * d + j] * S[(size_t)i * d + j];
    nc[i] = std::sqrt(a); nd[i] = std::sqrt(b);
  }
  double lcos = 0.0;
  for (int64_t q = 0; q < P; ++q) {
    const double* f = F + (size_t)q * d;
    double fc = 0.0, fd = 0.0;
    for (int j = 0; j < d_clip; ++j) fc += f[j] * f[j];
    for (int j = d_clip; j < d; ++j) fd += f[j] * f[j];
    fc = std::sqrt(fc); fd = std::sqrt(fd);
    int best = 0;
    double cbest = 0.0, dbest = 0.0;
    for (int i = 0; i < N; ++i) {
      double a = 0.0, b = 0.0;
      for (int j = 0; j < d_clip; ++j) a += f[j] * S[(size_t)i * d + j];
      for (int j = d_clip; j < d; ++j) b += f[j] * S[(size_t)i * d + j];
      const double cc = a / (fc * nc[i]), cd = b / (fd * nd[i]);
      D[i] = cc + lambda_dino * cd;
      if (i == 0 || D[i] > D[best]) { best = i; cbest = cc; dbest = cd; }
    }
    double second = -std::numeric_limits<double>::infinity();
    for (int i = 0; i < N; ++i) if (i != best) second = std::max(second, D[i]);
    if (index) index[q] = best;
    if (gap) gap[q] = N > 1 ? D[best] - second : std::numeric_limits<double>::infinity();
    rr[best] += 1.0;
    double mx = D[best], Z = 0.0;
    for (int i = 0; i < N; ++i) Z += std::exp(D[i] - mx);
    for (int i = 0; i < N; ++i) pp[i] += std::exp(D[i] - mx) / Z;
    lcos += (1.0 - cbest) + lambda_dino * (1.0 - dbest);
    if (scores) for (int i = 0; i < N; ++i) scores[(size_t)q * N + i] = D[i];
  }
  double llb = 0.0;
  for (int i = 0; i < N; ++i) {
    rr[i] /= (double)P; pp[i] /= (double)P;
    llb += rr[i] * pp[i];
    if (r) r[i] = rr[i];
    if (p) p[i] = pp[i];
  }
  if (loss) { loss[0] = lcos / (double)P; loss[1] = llb; loss[2] = lambda_cos * loss[0] + lambda_lb * loss[1]; }
  return 0;
}

}  // extern "C"

// ===================================================================================================
// Adaptive spatial smoothing (SURVEY.md 8(f) item 3; PAPER.md:149-157 Eq. 13-14, :362-370 Table 4).
extern "C" {

// s_MLP = MLP(PE(p)) (Eq. 13): PE of frequency 0 is the identity on the 3 coordinates (Table 4: "PE config 0, out size
// 3"); MLP = n_layers fully connected layers, ReLU after all but the last (Table 4: 3 -> 128 -> 128 -> 128 -> 8).
// L_smo = mean_i [ |s_MLP,i - sg(s_i)|_2 + max(sg(u_i), w_s) |sg(s_MLP,i) - s_i|_2 ]   (Eq. 14 read as SURVEY.md C-23;
// reading C-25: Euclidean norms as printed, not squared; mean over the n Gaussians; sg = stop gradient).
// Reverse mode, all fp64, one Gaussian at a time: with e = s_MLP - s, rho = |e|_2 (gradient 0 at rho = 0):
//   dL/ds_MLP = e / (n rho)   (first term only)   -> dW_l, db_l through the MLP;   no gradient reaches p (reading C-25:
//   "the optimizing of these semantic parameters does not affect original reconstruction quality");
//   dL/ds = -max(u, w_s) e / (n rho)   (second term only);   dL/du = 0.
// p [n][dims[0]], s [n][dims[L]], u [n]; W_l [dims[l+1]][dims[l]], b_l [dims[l+1]] or NULL.
// Outputs: loss[0] = L_smo; s_mlp [n][dims[L]] (optional); ds [n][dims[L]] (overwritten); dW_l, db_l ADDED to.
int oracle_smooth_loss(int64_t n, int n_layers, const int32_t* dims, const double* p, const double* s, const double* u,
                       const double* const* W, const double* const* b, double w_s, double* loss, double* s_mlp, double* ds,
                       double* const* dW, double* const* db) {
  if (n_layers < 1 || n_layers > 8 || n < 1) return -1;
  const int Fo = dims[n_layers];
  std::vector<std::vector<double>> act(n_layers + 1), pre(n_layers + 1), g(n_layers + 1);
  double total = 0.0;
  for (int64_t i = 0; i < n; ++i) {
    act[0].assign(p + (size_t)i * dims[0], p + (size_t)(i + 1) * dims[0]);
    for (int l = 0; l < n_layers; ++l) {
      const int in = dims[l], out = dims[l + 1];
      pre[l + 1].assign((size_t)out, 0.0);
      act[l + 1].assign((size_t)out, 0.0);
      for (int o = 0; o < out; ++o) {
        double a = (b && b[l]) ? b[l][o] : 0.0;
        for (int k = 0; k < in; ++k) a += W[l][(size_t)o * in + k] * act[l][k];
        pre[l + 1][o] = a;
        act[l + 1][o] = (l + 1 < n_layers && a < 0.0) ? 0.0 : a;
      }
    }
    double rho2 = 0.0;
    for (int f = 0; f < Fo; ++f) {
      const double e = act[n_layers][f] - s[(size_t)i * Fo + f];
      rho2 += e * e;
      if (s_mlp) s_mlp[(size_t)i * Fo + f] = act[n_layers][f];
    }
    const double rho = std::sqrt(rho2), wgt = std::max(u[i], w_s);
    total += rho + wgt * rho;
    g[n_layers].assign((size_t)Fo, 0.0);
    for (int f = 0; f < Fo; ++f) {
      const double e = act[n_layers][f] - s[(size_t)i * Fo + f];
      const double dir = rho > 0.0 ? e / rho : 0.0;
      g[n_layers][f] = dir / (double)n;
      ds[(size_t)i * Fo + f] = -wgt * dir / (double)n;
    }
    for (int l = n_layers - 1; l >= 0; --l) {
      const int in = dims[l], out = dims[l + 1];
      if (l + 1 < n_layers)
        for (int o = 0; o < out; ++o) if (!(pre[l + 1][o] > 0.0)) g[l + 1][o] = 0.0;
      g[l].assign((size_t)in, 0.0);
      for (int o = 0; o < out; ++o) {
        const double go = g[l + 1][o];
        if (db && db[l]) db[l][o] += go;
        for (int k = 0; k < in; ++k) {
          dW[l][(size_t)o * in + k] += go * act[l][k];
          g[l][k] += W[l][(size_t)o * in + k] * go;
        }
      }
    }
  }
  loss[0] = total / (double)n;
  return 0;
}

}  // extern "C"

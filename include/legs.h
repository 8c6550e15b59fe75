/* legs.h — C-ABI of the B200-native hot path of "Language Embedded 3D Gaussians" (arxiv 2311.18482).
 *
 * What the calls compute (citations are PAPER.md lines + the reading in DESIGN.md where the paper is silent):
 *   legs_preprocess        per-Gaussian projection for I = R(p, Sigma, c, alpha; p_cam)   PAPER.md:56-58 (Eq. 1); C-1..C-12
 *   legs_bin_and_sort      tile lists: (tile<<32 | depth) keys, stable radix sort, ranges  BASELINE.json north_star (2); C-7, C-8
 *   legs_render_forward    alpha blending of colour, s_G (R_s) and u (R_u)                 PAPER.md:116-122 (Eq. 8), :138 (Eq. 10); C-9, C-10, C-13
 *   legs_render_backward   reverse mode of the above down to the 3D parameters             PAPER.md:56, :182; C-14..C-16
 *   legs_decode_semantics  M = softmax(D_MLP(R_s)), F = M . S                              PAPER.md:118-122 (Eq. 8), :333-358 (Eq. 21-22, Table 3)
 *   legs_relevancy         cosine of F[:, 0:d_clip] against query vectors                  PAPER.md:360; C-21
 *
 * Conventions
 *   - Every data pointer is a DEVICE pointer owned by the caller, 16-byte aligned, valid until the work enqueued on
 *     `stream` has completed. Structs (legs_camera, legs_gaussians, ...) are HOST structs passed by pointer and
 *     copied by value at call time. The library never allocates or frees device memory and never synchronises,
 *     except legs_read_num_instances (one stream sync).
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream). All work of one call is enqueued
 *     on that stream in order.
 *   - Every function returns 0 (LEGS_OK) or a negative legs_status. Argument errors are detected synchronously and
 *     nothing is enqueued. The one data-dependent error (more tile instances than `capacity`) is reported through
 *     bit 63 of *frame->num_instances and returned by legs_read_num_instances.
 *   - Activations (exp on scales, sigmoid on opacity, quaternion normalisation) are the caller's (reading C-3);
 *     gradients are with respect to the activated values.
 *   - Camera: looks down +z, x right, y down; principal point in continuous image coordinates, pixel (i,j) is
 *     sampled at (i,j) in the pixel-index space used by mean2d (C-4).
 */
#ifndef LEGS_H_
#define LEGS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  LEGS_OK = 0,
  LEGS_ERR_NULL = -1,      /* a required pointer is NULL */
  LEGS_ERR_ALIGN = -2,     /* a device pointer is not 16-byte aligned */
  LEGS_ERR_DIM = -3,       /* a size / dimension argument is out of range */
  LEGS_ERR_CAPACITY = -4,  /* tile instances exceed the capacity given to legs_bin_and_sort */
  LEGS_ERR_WORKSPACE = -5, /* workspace too small (see the *_workspace_bytes queries) */
  LEGS_ERR_CUDA = -6       /* a CUDA runtime call failed (legs_last_cuda_error gives the code) */
} legs_status;

typedef struct legs_ctx legs_ctx;

/* Creates a context for CUDA device `device` (host-side metadata only: SM count, kernel attributes). */
int legs_create(int device, legs_ctx** out);
void legs_destroy(legs_ctx* ctx);
const char* legs_status_string(int status);
int legs_last_cuda_error(const legs_ctx* ctx);
/* Number of kernels this context has launched since creation (for bench.py's gpu_launches). */
uint64_t legs_launch_count(const legs_ctx* ctx);

#define LEGS_TILE 16            /* tile edge in pixels (north_star (2), configs[0]) */
#define LEGS_MAX_SEM_DIM 32

typedef struct {
  int32_t width, height;
  float fx, fy, cx, cy;
  float world_to_cam[12]; /* row-major 3x4 [R|t] */
  float near_plane;       /* cull if z_view <= near_plane (0.2 in every config) */
  float background[3];    /* added to rgb as T_final * background; sem/unc/depth get none (C-10) */
} legs_camera;

typedef struct {
  int64_t n;
  int32_t sh_degree;       /* 0..3 active degree */
  int32_t sh_coefs_stored; /* coefficients per channel in `sh` (>= (sh_degree+1)^2) */
  int32_t sem_dim;         /* F: multiple of 4, 4..32 */
  const float* means;      /* [n,3] world */
  const float* scales;     /* [n,3] > 0 */
  const float* quats;      /* [n,4] (w,x,y,z), unit; not normalised inside (C-2) */
  const float* opacities;  /* [n] in (0,1) */
  const float* sh;         /* [n, sh_coefs_stored, 3] */
  const float* sem;        /* [n,F] compact semantic feature s_G */
  const float* unc;        /* [n] uncertainty u in [0,1] */
} legs_gaussians;

/* Per-view, per-Gaussian results of legs_preprocess. All arrays have n entries (rows). Culled Gaussians have
 * tiles_touched = 0, radius = 0, rect = 0 and zeros elsewhere, except depth which always holds z_view. */
typedef struct {
  float* depth;            /* [n] view-space z */
  int32_t* radius;         /* [n] ceil(3 sqrt(lambda_max)) */
  int32_t* rect;           /* [n,4] x0,y0,x1,y1 in tiles, x1/y1 exclusive */
  float* mean2d;           /* [n,2] pixel-index space */
  float* conic_opacity;    /* [n,4] A,B,C,opacity */
  float* rgb;              /* [n,3] clamped at 0 */
  uint8_t* clamped;        /* [n] bit0..2: rgb channel clamped; bit3/4: Jacobian x/y clamp active */
  uint32_t* tiles_touched; /* [n] */
  float* record;           /* [n, legs_record_stride(F)] packed compositor record (rows of culled Gaussians are
                              not written): mu_x, mu_y, r11, r12, r22, opacity, r, g, b, depth, sem[F], u, thr.
                              (r11, r12, r22) = sqrt(log2(e)/2) * upper Cholesky factor of the conic, so that
                              exp(-1/2 d^T Q d) = 2^-((r11 dx + r12 dy)^2 + (r22 dy)^2); thr = log2(255 opacity)
                              (+ margin), the compositors' cull threshold on that exponent */
  uint64_t* num_instances; /* device scalar D = sum tiles_touched; bit 63 set by legs_bin_and_sort on overflow */
} legs_frame;

int32_t legs_record_stride(int32_t sem_dim);  /* floats per record: roundup4(11 + F) */
int32_t legs_pixel_channels(int32_t sem_dim); /* CH = roundup4(3 + 1 + F + 1 + 1) */
size_t legs_sort_workspace_bytes(int64_t n, uint64_t capacity, int32_t width, int32_t height);
size_t legs_backward_workspace_bytes(int64_t n, int32_t sem_dim);

/* S1: projection of every Gaussian; D = sum of tiles_touched is reduced into *frame->num_instances. */
int legs_preprocess(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam, legs_frame* frame, void* stream);

/* Copies D to the host after synchronising `stream`. Returns LEGS_ERR_CAPACITY if bit 63 is set. */
int legs_read_num_instances(legs_ctx* ctx, const legs_frame* frame, uint64_t* host_out, void* stream);

/* S2 + S3 + S4: tile lists in ascending (tile, depth bits, index) order and per-tile ranges. The result is the one a
 * stable sort of the 64-bit keys (tile << 32 | float_bits(depth)), emitted in index order, would give. It is reached
 * without any pass over the D tile instances: the n Gaussians are radix-sorted by depth bits; per-tile counts (hence
 * `ranges` and D) come from a 2D difference array of the tile rects; one entry per (Gaussian, tile ROW of its rect) is
 * emitted, by a ranked pass over the depth-ordered Gaussians, straight into (row, depth) order; the row entries are then
 * expanded into the tile lists, one 4-byte write per instance.
 * Launches are sized for `capacity`; n and capacity must be below 2^30; kernels read D on the device (the exact 64-bit
 * count of legs_preprocess decides the overflow test, so it is also detected when D exceeds 2^32). keys_sorted [capacity] (optional, may be
 * NULL) receives the 64-bit keys; vals_sorted [capacity] and ranges [tiles,2] are required.
 * ranges[t] = [first, last+1) in the sorted arrays, (0,0) for an empty tile. */
int legs_bin_and_sort(legs_ctx* ctx, const legs_frame* frame, const legs_camera* cam, int64_t n, uint64_t capacity,
                      uint64_t* keys_sorted, uint32_t* vals_sorted, uint32_t* ranges, void* workspace,
                      size_t workspace_bytes, void* stream);

/* S5: out_pixels [H,W,CH]: 0-2 rgb, 3 depth (sum w z), 4..4+F-1 sem, 4+F unc, 5+F alpha = 1 - T_final;
 * slot 6+F holds the final transmittance T_final (read back by legs_render_backward), slot 7+F is 0.
 * n_contrib [H,W]: 1-based position in the tile list of the last blended Gaussian (0 = none).
 * sem_bf16 [H*W, F] (optional, may be NULL): bf16 copy of the semantic channels for legs_decode_semantics.
 * block_masks [capacity] (optional, may be NULL): one byte per tile-list position, written for the entries the tile's
 * compositor staged: which of the tile's eight 8x4-pixel warp blocks the Gaussian can reach (alpha >= 1/255). Passing the
 * same buffer to legs_render_backward saves it the recomputation; it has no meaning outside that hand-over. */
int legs_render_forward(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam, const legs_frame* frame,
                        const uint32_t* vals_sorted, const uint32_t* ranges, float* out_pixels, uint32_t* n_contrib,
                        uint16_t* sem_bf16, uint8_t* block_masks, void* stream);

/* Measurement variant of legs_render_forward: identical outputs, and counters[0..3] (device, caller-zeroed, uint64)
 * += pixel-Gaussian pairs the kernel examines (after its block culling), blended pairs, tile-list entries staged, and
 * the pairs a plain per-tile walk examines (every list entry up to each pixel's termination point: the P_e of
 * SURVEY.md 8(d)). Used by bench.py for the ALU rooflines. */
int legs_render_forward_stats(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam, const legs_frame* frame,
                              const uint32_t* vals_sorted, const uint32_t* ranges, float* out_pixels,
                              uint32_t* n_contrib, uint64_t* counters, void* stream);

typedef struct {
  float* dmeans;     /* [n,3] */
  float* dscales;    /* [n,3] */
  float* dquats;     /* [n,4] */
  float* dopacities; /* [n] */
  float* dsh;        /* [n, sh_coefs_stored, 3] */
  float* dsem;       /* [n,F] */
  float* dunc;       /* [n] */
  float* dmean2d;    /* [n,2] dL/dmean2d in pixels (C-16) */
} legs_grads;

#define LEGS_BWD_ACCUMULATE 1 /* add into grads instead of overwriting */
#define LEGS_BWD_COUPLE_SEM 2 /* sem/unc upstream gradients also flow to alpha/geometry (C-14); default: only to dsem/dunc */
#define LEGS_BWD_COMPOSITE_ONLY 4 /* measurement only: run S6 (the compositor) and stop before S7; grads are not written */
#define LEGS_BWD_DEPTH_ALPHA 8 /* the depth slot (3) and the alpha slot (5+F) of dL_dpixels are read too (SURVEY.md 8(f) item
                                  4, reading C-17b): depth_out = sum w z is one more blended channel whose value z = t_z
                                  reaches the means; alpha_out = 1 - T_final gives d alpha_out / d alpha_k = T_final / (1 - alpha_k) */

/* S6 + S7. dL_dpixels [H,W,CH]: rgb, sem and unc slots are read; depth/alpha slots only with LEGS_BWD_DEPTH_ALPHA (C-17),
 * pad slots never.
 * out_pixels and n_contrib (and block_masks, optional: NULL = recompute) are the outputs of legs_render_forward for the
 * same frame. */
int legs_render_backward(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam, const legs_frame* frame,
                         const uint32_t* vals_sorted, const uint32_t* ranges, const float* out_pixels,
                         const uint32_t* n_contrib, const float* dL_dpixels, const uint8_t* block_masks, int32_t flags,
                         legs_grads* grads, void* workspace, size_t workspace_bytes, void* stream);

/* Launch order for the compositors: tile_order [n_tiles] u32 (device, caller-owned) receives the tile indices with the
 * longest lists first (bucketed by list length, four buckets per octave; the order inside a bucket is unspecified).
 * ranges [n_tiles,2] is the output of legs_bin_and_sort for the same frame; n_tiles = ceil(W/16) ceil(H/16) <= 2^22.
 * The *_ordered forms of the two render calls take it as one more argument: CTA b then works on tile tile_order[b] instead of
 * tile b. Results do not depend on the order (forward: bit-identical; backward: the same sums, accumulated by atomics as
 * before); it only shortens the tail of the launch when a few tiles hold very long lists (clustered scenes: configs[4]).
 * tile_order = NULL is the plain call. The array must be a permutation of 0..n_tiles-1 for the camera of the render call. */
int legs_tile_order(legs_ctx* ctx, const uint32_t* ranges, int32_t n_tiles, uint32_t* tile_order, void* stream);
int legs_render_forward_ordered(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam, const legs_frame* frame,
                                const uint32_t* vals_sorted, const uint32_t* ranges, float* out_pixels, uint32_t* n_contrib,
                                uint16_t* sem_bf16, uint8_t* block_masks, const uint32_t* tile_order, void* stream);
int legs_render_backward_ordered(legs_ctx* ctx, const legs_gaussians* g, const legs_camera* cam, const legs_frame* frame,
                                 const uint32_t* vals_sorted, const uint32_t* ranges, const float* out_pixels,
                                 const uint32_t* n_contrib, const float* dL_dpixels, const uint8_t* block_masks,
                                 int32_t flags, legs_grads* grads, void* workspace, size_t workspace_bytes,
                                 const uint32_t* tile_order, void* stream);

typedef struct {
  int32_t n_layers;     /* 2 or 3 linear layers, ReLU between, none after the last */
  int32_t in_dim;       /* 8 or 16 */
  int32_t hidden[2];    /* hidden widths (hidden[1] unused when n_layers == 2); multiples of 16, <= 256 */
  int32_t n_codes;      /* K: 32, 64 or 128 */
  const uint16_t* w[3]; /* bf16 [out,in] row-major */
  const float* b[3];    /* fp32 [out] or NULL */
} legs_decoder;

size_t legs_decode_workspace_bytes(const legs_decoder* dec, int32_t d);

/* S9 + S10: probs = softmax(MLP(feat)) [P,K] bf16 (optional), decoded = probs . codebook [P,d] bf16 (optional).
 * feat [P,in_dim] bf16; codebook [K,d] bf16, d multiple of 64, d <= 1024. bf16 operands, fp32 accumulation. */
int legs_decode_semantics(legs_ctx* ctx, const uint16_t* feat, int64_t P, const legs_decoder* dec,
                          const uint16_t* codebook, int32_t d, uint16_t* probs, uint16_t* decoded, void* workspace,
                          size_t workspace_bytes, void* stream);

/* The two halves of legs_decode_semantics, for inference over many frames with fixed weights: legs_decode_prepare packs
 * the decoder weights and the codebook into `workspace` once; legs_decode_semantics_packed is the per-frame call
 * (same outputs, no packing launch). */
int legs_decode_prepare(legs_ctx* ctx, const legs_decoder* dec, const uint16_t* codebook, int32_t d, void* workspace,
                        size_t workspace_bytes, void* stream);
int legs_decode_semantics_packed(legs_ctx* ctx, const uint16_t* feat, int64_t P, const legs_decoder* dec, int32_t d,
                                 uint16_t* probs, uint16_t* decoded, const void* workspace, size_t workspace_bytes,
                                 void* stream);

/* S11: rel[p,q] = <F_p[0:d_clip], query_q> / (|F_p[0:d_clip]| |query_q|) with F = probs . codebook, computed from
 * probs [P,K] bf16 without materialising F (Gram shortcut). queries [Q,d_clip] bf16, Q <= 16, d_clip <= min(d, 1024);
 * rel [P,Q] fp32.
 * workspace: legs_relevancy_workspace_bytes(K, Q). */
size_t legs_relevancy_workspace_bytes(int32_t K, int32_t Q);
int legs_relevancy(legs_ctx* ctx, const uint16_t* probs, int64_t P, const uint16_t* codebook, int32_t K, int32_t d,
                   int32_t d_clip, const uint16_t* queries, int32_t Q, float* rel, void* workspace,
                   size_t workspace_bytes, void* stream);
/* The same in two halves: legs_relevancy_prepare packs the Gram matrix S_c S_c^T and S_c q / |q| once per codebook and
 * query set (K in {32, 64, 128}, Q <= 16, d_clip <= min(d, 1024)); legs_relevancy_packed is the per-frame call. */
int legs_relevancy_prepare(legs_ctx* ctx, const uint16_t* codebook, int32_t K, int32_t d, int32_t d_clip,
                           const uint16_t* queries, int32_t Q, void* workspace, size_t workspace_bytes, void* stream);
int legs_relevancy_packed(legs_ctx* ctx, const uint16_t* probs, int64_t P, int32_t K, int32_t Q, float* rel,
                          const void* workspace, size_t workspace_bytes, void* stream);

/* S11 from an already decoded map (the `input_is_probs = 0` case of legs_relevancy; "the
 * relevance map of F", reading C-21): rel[p,q] = <F_p[0:d_clip], query_q> / (|F_p[0:d_clip]| |query_q|) for a caller that
 * holds only F = decoded [P,d] bf16 (row pitch d; the `decoded` output of legs_decode_semantics) and no probabilities.
 * queries [Q,d_clip] bf16 (need not be unit vectors), Q <= 16; d and d_clip multiples of 8, 8 <= d_clip <= min(d, 1024);
 * rel [P,Q] fp32. A row of F that is all zero in its first d_clip entries gives 0. No workspace. Streams F once
 * (2 d_clip bytes per pixel); legs_relevancy from the probabilities reads 2 K bytes per pixel instead and is the cheaper
 * call whenever the probabilities exist. */
int legs_relevancy_decoded(legs_ctx* ctx, const uint16_t* decoded, int64_t P, int32_t d, int32_t d_clip,
                           const uint16_t* queries, int32_t Q, float* rel, void* stream);

/* legs_relevancy without caller scratch, for callers that cannot allocate device memory. Some users of this library run
 * where cudaMalloc is off limits: a real-time viewer or serving loop that took all its memory from a pool at start-up (an
 * allocation in the frame loop can synchronise the device and stall every stream), a plugin that only receives the host
 * application's input and output buffers and has no allocator of its own, or a job whose memory budget is already spent.
 * For them the 32-64 KB that legs_relevancy packs the Gram matrix and the projected queries into live in a fixed array
 * inside the library instead of in a `workspace` argument. Same arguments otherwise, same kernels, same results.
 *   - Limit: K <= legs_relevancy_static_max_codes() = 128 (and K in {32, 64, 128}, Q <= 16, d_clip <= min(d, 1024) as for
 *     legs_relevancy); anything larger returns LEGS_ERR_DIM and nothing is enqueued. The array is
 *     legs_relevancy_static_bytes() = 64 KB on EVERY GPU that loads the library, held until the process exits.
 *   - The call allocates and frees nothing, and calls no library routine that does. The first call on each device looks
 *     up the array's device address (a host-side runtime query, no device work); make that first call with the context's
 *     device current and before any stream capture begins. Later calls only enqueue work on `stream`.
 *   - The device that is current at the call must be the context's device (else LEGS_ERR_CUDA, invalid device).
 *   - All calls on one device share the one array, and it keeps what the last call packed. Each call clears and repacks
 *     the part it uses, so results never depend on earlier calls; but two calls whose GPU work can overlap (different
 *     streams, or several host threads, without an ordering between them) race on it and give undefined relevancies.
 *     Issue them on one stream, or order them with events. */
size_t legs_relevancy_static_bytes(void);
int32_t legs_relevancy_static_max_codes(void);
int legs_relevancy_static(legs_ctx* ctx, const uint16_t* probs, int64_t P, const uint16_t* codebook, int32_t K, int32_t d,
                          int32_t d_clip, const uint16_t* queries, int32_t Q, float* rel, void* stream);

/* LERF-style relevancy (optional). PAPER.md:360 computes the relevancy map "in accordance with LERF
 * [18]" without giving the formula (reading C-21b: by this paper the function is "parity unpinned"; it restates LERF's
 * published score). cosines [P,Q] fp32 = the output of legs_relevancy for Q query vectors of which the first n_pos are the
 * user's queries and the remaining Q - n_pos are canonical negative phrases:
 *   out[p][j] = min_i exp(tau c_pj) / (exp(tau c_pj) + exp(tau c_pi)),  j < n_pos <= i < Q   (out [P,n_pos] fp32).
 * 2 <= Q <= 16, 1 <= n_pos < Q, 0 <= tau <= 100 (LERF uses 10). */
int legs_relevancy_lerf(legs_ctx* ctx, const float* cosines, int64_t P, int32_t Q, int32_t n_pos, float tau, float* out,
                        void* stream);

/* ---- widening: the semantic loss head between legs_render_forward and legs_render_backward.
 * M^ = softmax(D_MLP(R_s)) (Eq. 8); L_CE = sum_p CE(M^_p, M_p) (1 - R_u,p) / P (Eq. 10, CE = -log M^_p[m],
 * natural logarithm); L_u = sum_p R_u,p / P (Eq. 11); L_s = lambda_ce L_CE + lambda_u L_u (Eq. 12); and its reverse mode
 * down to the rendered maps and the decoder weights. First layer and softmax in fp32, the other contractions on the
 * tensor cores with bf16 operands and fp32 accumulation.
 * Decoders: 2 layers with in_dim = sem_dim in {8, 16}, hidden[0] in {32, 64}; or the paper's Table 3 shape
 * (PAPER.md:344-351), 3 layers sem_dim -> 128 -> 256 -> n_codes; n_codes in {32, 64, 128} (else LEGS_ERR_DIM). */
typedef struct {
  float* dw[3]; /* fp32 [out,in] per layer, ADDED to (the caller zeroes them; lets several views accumulate) */
  float* db[3]; /* fp32 [out] per layer or NULL, added to */
} legs_decoder_grads;

/* Workspace of legs_semantic_loss for P pixels. 2-layer decoders: 24 KB of packed weights. 3-layer decoders: 144 KB of
 * packed weights + 768 B per pixel (rounded up to 128-pixel tiles): the bf16 operand tiles of the middle layer's weight
 * gradient, written by the main kernel and read back by a streaming kernel (both weight-gradient accumulators of that
 * shape do not fit in tensor memory at once). */
size_t legs_loss_workspace_bytes(const legs_decoder* dec, int64_t P);

/* pixels [P,CH] fp32: the out_pixels of legs_render_forward (R_s in slots 4..4+F-1, R_u in slot 4+F are read).
 * index_map [P] int32: the discrete semantic index m of every pixel, in [0, n_codes).
 * dL_dpixels [P,CH]: slots 4..4+F-1 receive dL_s/dR_s and slot 4+F receives dL_s/dR_u (overwritten; the other slots
 * are left as they are), ready to be passed to legs_render_backward.
 * loss [3] fp32 device: L_CE, L_u, L_s are ADDED to it (the caller zeroes it). */
int legs_semantic_loss(legs_ctx* ctx, const float* pixels, int64_t P, int32_t sem_dim, const int32_t* index_map,
                       const legs_decoder* dec, float lambda_ce, float lambda_u, float* dL_dpixels,
                       const legs_decoder_grads* grads, float* loss, void* workspace, size_t workspace_bytes, void* stream);

/* ---- widening: quantisation search and codebook losses, PAPER.md:76-108 (Eq. 3-7), :310-329
 * (Eq. 16-20). features [P,d] bf16 = hybrid language features F = F^CLIP (+) F^DINO (Eq. 2: the first d_clip dims are the
 * CLIP part); codebook [N,d] bf16 = the discrete feature space S. Computes, on the tensor cores (bf16 x bf16, fp32 acc):
 *   D(F, f_i) = cos<F^CLIP, f_i^CLIP> + lambda_dino cos<F^DINO, f_i^DINO> (Eq. 4);  index_map[p] = argmax_i D (Eq. 16; ties go
 *   to the lowest index, reading C-28);  r = sum onehot(m) / P (Eq. 17);  p = sum softmax_i(D) / P (Eq. 18-19);
 *   loss[0] = L_cos = mean over the P features of (1 - cos_CLIP(m)) + lambda_dino (1 - cos_DINO(m)) (Eq. 5, reading C-29);
 *   loss[1] = L_lb = sum_i r_i p_i (Eq. 20);  loss[2] = L_q = lambda_cos L_cos + lambda_lb L_lb (Eq. 7).
 * N in {32, 64, 128}; d and d_clip multiples of 64, 64 <= d_clip < d <= 4096; 0 <= lambda_dino <= 8.
 * index_map [P] int32; r, p [N] fp32 (optional, may be NULL); loss [3] fp32 device (overwritten).
 * The gradient of L_q with respect to the codebook is not part of this call. */
size_t legs_quantize_workspace_bytes(int32_t N);
int legs_quantize(legs_ctx* ctx, const uint16_t* features, int64_t P, const uint16_t* codebook, int32_t N, int32_t d,
                  int32_t d_clip, float lambda_dino, float lambda_cos, float lambda_lb, int32_t* index_map, float* r,
                  float* p, float* loss, void* workspace, size_t workspace_bytes, void* stream);

/* ---- widening: adaptive spatial smoothing, PAPER.md:149-157 (Eq. 13-14), :362-370 (Table 4).
 *   s_MLP = MLP(PE(p)) (Eq. 13): PE of frequency 0 = the 3 coordinates; MLP = 3 -> hidden -> hidden -> hidden -> sem_dim, ReLU after
 *   the first three layers (Table 4; hidden = 128 in this version).
 *   L_smo = mean_i [ |s_MLP,i - sg(s_i)|_2 + max(sg(u_i), w_s) |sg(s_MLP,i) - s_i|_2 ]  (Eq. 14, readings C-23 / C-25; sg = stop
 *   gradient; w_s = 0.1 at PAPER.md:182).
 * Forward and reverse mode in one call: loss[0] += L_smo (unscaled); dsem [n,F] = (or +=, if `accumulate`) lambda_smo dL_smo/ds;
 * grads->dw[l] / db[l] += lambda_smo dL_smo/dW_l, db_l (fp32, the caller zeroes them; db entries may be NULL). No gradient
 * reaches the positions or the uncertainties (reading C-25). Layers 2 and 3 and every weight gradient run on the tensor
 * cores with bf16 operands and fp32 accumulation; the first and last layer and the loss in fp32. */
typedef struct {
  int32_t hidden;       /* 128 */
  const uint16_t* w[4]; /* bf16 [out,in] row-major: [hidden,3], [hidden,hidden], [hidden,hidden], [sem_dim,hidden] */
  const float* b[4];    /* fp32 [out] or NULL */
} legs_smooth_mlp;
typedef struct {
  float* dw[4]; /* fp32 [out,in], added to */
  float* db[4]; /* fp32 [out] or NULL, added to */
} legs_smooth_grads;
size_t legs_smooth_workspace_bytes(int32_t sem_dim);
int legs_smooth_loss(legs_ctx* ctx, int64_t n, int32_t sem_dim, const float* means, const float* sem, const float* unc,
                     const legs_smooth_mlp* mlp, float w_s, float lambda_smo, int32_t accumulate, float* dsem,
                     const legs_smooth_grads* grads, float* loss, void* workspace, size_t workspace_bytes, void* stream);

/* ---- widening: training-step plumbing named at PAPER.md:182.
 * legs_adam_step: one Adam step (Kingma & Ba [25], Algorithm 1 with bias correction; lr 1e-3, betas
 * (0.9, 0.999); eps is the caller's, reading C-26: 1e-8) over up to 16 parameter tensors in ONE launch, in place:
 *   m <- b1 m + (1-b1) g;  v <- b2 v + (1-b2) g^2;  p <- p - lr (m / (1-b1^t)) / (sqrt(v / (1-b2^t)) + eps).
 * params / grads / m / v: HOST arrays of n_tensors DEVICE pointers (fp32, 16-byte aligned, counts[t] floats each).
 * The gradients are those of legs_render_backward / legs_semantic_loss (w.r.t. the values passed to the library). */
typedef struct {
  float lr, beta1, beta2, eps;
  int32_t step; /* t, 1-based */
} legs_adam;
int legs_adam_step(legs_ctx* ctx, int32_t n_tensors, float* const* params, const float* const* grads, float* const* m,
                   float* const* v, const int64_t* counts, const legs_adam* hp, void* stream);

/* Density-control statistics of one view ("adaptive density control" following [17]; reading C-27): for
 * every Gaussian with radius[i] > 0 (visible in the view that produced them): grad_accum[i] += |dmean2d[i]|_2 (pixels),
 * denom[i] += 1, max_radius[i] = max(max_radius[i], radius[i]). dmean2d [n,2] is legs_grads.dmean2d of that view (not
 * accumulated over views), radius [n] is legs_frame.radius. */
int legs_density_stats(legs_ctx* ctx, int64_t n, const float* dmean2d, const int32_t* radius, float* grad_accum,
                       uint32_t* denom, int32_t* max_radius, void* stream);

/* ---- measurement (the FP32 and MUFU peaks the ALU rooflines divide by are measured in the bench run).
 * Launches one micro-benchmark kernel on `stream` (num_sms x 8 CTAs of 256 threads, 8 independent chains per thread):
 * kind 0 = fma.rn.f32 chains, 1 = ex2.approx chains, 2 = packed fma.rn.f32x2 chains, 3 = FMA + warp shuffle mix.
 * sink: device buffer of num_sms * 8 * 256 floats (never written in practice). *lane_ops_host (HOST pointer) receives
 * the number of FMA / ex2 lane-operations the launch executes; the caller times the launch with events. */
int legs_peak_kernel(legs_ctx* ctx, int32_t kind, int32_t iters, float* sink, uint64_t* lane_ops_host, void* stream);
int32_t legs_num_sms(const legs_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* LEGS_H_ */

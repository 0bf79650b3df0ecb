/* gs.h -- C-ABI of the B200-native differentiable 3D Gaussian Splatting rasteriser (libgs.so).
 *
 * What is wrapped (arxiv/paper_2605_10760, MAGS-SLAM): the renderer behind per-agent mapping (Eq. 4),
 * the per-keyframe pose deltas and the joint refinement of the fused map (Eq. 23): Gaussians with
 * centre mu, scale s, rotation q, opacity and colour (Eq. 19), a pinhole camera
 * (f_x,f_y,c_x,c_y) with a WORLD-TO-CAMERA SE(3) pose T_k, "the differentiably rendered
 * RGB and depth" plus alpha, and the gradients w.r.t. every Gaussian parameter and the pose.
 * The paper does not specify the rasteriser; constants and conventions are the readings Q1-Q17 of DESIGN.md.
 *
 * One iteration is the call sequence
 *     gs_preprocess -> gs_bin_tiles -> gs_rasterize_fwd -> [caller forms dL/dRGB, dL/dDepth] -> gs_rasterize_bwd
 *     -> gs_pose_grad (optional)
 * Every step runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.
 *
 * Conventions common to all calls
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All work is enqueued on it and
 *     the calls return without synchronising, except where stated.
 *   - Array arguments are caller-owned, contiguous DEVICE pointers on the context's device unless marked HOST.  They
 *     must stay valid until the stream has executed the work.  The library never frees or reallocates them.
 *     gs_preprocess RETAINS the parameter pointers (means ... sh, T_cw_dev) until the gs_rasterize_bwd / gs_pose_grad
 *     of the same iteration, which re-read them.
 *   - gs_ctx owns all scratch (features, keys, sorted lists, per-pixel state, 2-D gradients); it only grows.  A
 *     context is not thread-safe; use one context per stream.
 *   - Return value: 0 (GS_OK) or a negative gs_status.  gs_last_error() gives a context-owned message.  No call
 *     aborts, throws or prints.
 *   - Pixels are integer-centred: pixel (px,py) samples the image plane at (px,py)  (Q7).
 *   - Non-finite inputs are the caller's responsibility: a Gaussian whose projection is non-finite is culled.
 */
#ifndef GS_H_
#define GS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define GS_API __attribute__((visibility("default")))
#else
#define GS_API
#endif

typedef enum {
  GS_OK = 0,
  GS_E_INVALID = -1,  /* null pointer, bad size, bad degree */
  GS_E_ORDER = -2,    /* call sequence violated (e.g. gs_rasterize_bwd before gs_rasterize_fwd) */
  GS_E_CUDA = -3,     /* a CUDA runtime call failed; text in gs_last_error */
  GS_E_NOMEM = -4,    /* growing the scratch failed */
  GS_E_OVERFLOW = -5, /* the tile-instance capacity was exceeded by an asynchronous iteration: that iteration's outputs
                         are invalid (image = background, gradients = 0).  Reported once, by the first of
                         gs_preprocess / gs_bin_tiles / gs_poll / gs_get_counts to notice; the context has already
                         grown when it is returned: re-issue the iteration from gs_preprocess. */
  GS_E_TOO_LARGE = -6 /* a size beyond the fixed capacity of an entry point that owns no growable memory
                         (gs_compact_plan_static: N > gs_compact_plan_static_max()); nothing was launched */
} gs_status;

/* Pinhole camera + world-to-camera pose, p_c = R p_w + t.  HOST struct. */
typedef struct {
  int32_t width, height;
  float fx, fy, cx, cy;
  float near_z;    /* Gaussians with camera-space z <= near_z are culled (Q6); 0.2 in every config */
  float T_cw[12];  /* row-major 3x4 [R|t] */
} gs_camera;

typedef struct gs_ctx gs_ctx; /* opaque */

/* flags of gs_rasterize_bwd / gs_pose_grad */
#define GS_ACCUMULATE 1u /* parameter gradients are added to the output arrays instead of overwriting them (config 5);
                            the addition is one fp32 RED.ADD per element at L2 (a denormal sum is flushed to zero), so
                            several contexts on different streams may accumulate into the same arrays concurrently */
#define GS_POSE_ONLY 2u  /* Gaussians frozen: no parameter gradients are written; output pointers may be NULL (config 4) */
#define GS_SPARSE_GRADS 4u /* parameter gradients are written COMPACT: row r of every g_* array belongs to the Gaussian
                            gs_visible_ids()[r], r < n_visible (arrays need n_visible <= N rows); rows of culled Gaussians do
                            not exist (their gradient is zero), nothing is zero-filled.  What gs_adam_step_sparse consumes: the
                            dense (11 + 3K) N gradient write is 1/3 of the iteration's HBM bytes.  Not with GS_ACCUMULATE. */

/* Compile-time semantics of the rasteriser (DESIGN.md readings; north_star of BASELINE.json) */
#define GS_TILE 16               /* binning tiles are 16x16 pixels */
#define GS_ALPHA_MIN (1.0f / 255.0f) /* a Gaussian is skipped at a pixel iff alpha < 1/255           (Q1) */
#define GS_ALPHA_MAX 0.99f       /* alpha = min(0.99, opacity * G); no gradient through the clamp  (Q2) */
#define GS_T_MIN 1e-4f           /* a Gaussian is blended iff the transmittance in front of it >= 1e-4 (Q3) */
#define GS_DILATION 0.3f         /* Sigma' = J W Sigma W^T J^T + 0.3 I                              (Q4) */

/* Create / destroy a context on CUDA device `device`.  Synchronous. */
GS_API int gs_create(gs_ctx** out, int device);
GS_API int gs_destroy(gs_ctx* ctx);
/* Message of the last failing call on this context (never NULL; owned by the context). */
GS_API const char* gs_last_error(const gs_ctx* ctx);

/* Options of a context (take effect from the next gs_preprocess).
 *   GS_OPT_EXACT_TILE_CULL (default 0): gs_bin_tiles drops the (Gaussian, tile) instances whose ellipse {alpha >= 1/255}
 *   reaches no pixel region of the tile although the tile lies in the ellipse's bounding rectangle (the corner tiles of
 *   large footprints).  Images and gradients are unchanged (such instances never pass the alpha test); the per-tile lists
 *   become the (tile, depth, index)-ordered SUBSET of the default lists, so the mode sits outside the bit-exact binning
 *   contract: gs_get_counts still reports the rectangle-based instance total (the capacity the lists are laid out in),
 *   gs_get_binning's tile_ranges delimit the shorter lists and the entries between a list's end and the next list's
 *   start are unspecified. */
#define GS_OPT_EXACT_TILE_CULL 1
/*   GS_OPT_VIEW_STREAMS (default 1, 1..8): gs_refine_views issues its views round-robin on this context and on
 *     value - 1 context-owned sub-contexts with their own streams (forked from and joined to the caller's stream by
 *     events); every view then ACCUMULATES into gradient arrays zeroed up front.  The latency-bound per-Gaussian and
 *     binning kernels of one view overlap the compositing kernels of another (config 5: 164 -> 195 eight-view it/s at 4).
 *     Each sub-context holds its own scratch (about 250 bytes per Gaussian + 50 bytes per tile instance). */
#define GS_OPT_VIEW_STREAMS 2
GS_API int gs_set_option(gs_ctx* ctx, int option, int value);

/* Step a1 -- EWA projection, conic, screen extent, colour (oracle reading C1 steps 1-6, 8).
 *   N            number of Gaussians (0 <= N < 2^24: sorted list entries carry slot << 8 | region mask)
 *   sh_degree    0..3; K = (sh_degree+1)^2 coefficients per channel
 *   means        [N,3]  world-space centres mu
 *   scales       [N,3]  ACTIVATED scales s > 0  (Sigma = R diag(s)^2 R^T)
 *   quats        [N,4]  (w,x,y,z), any non-zero norm (normalised inside)
 *   opacities    [N]    ACTIVATED opacities in (0,1)
 *   sh           [N,K,3] real-SH coefficients, l-major / m = -l..l, RGB innermost; colour = max(0, sum_k B_k sh_k + 0.5)
 *   cam          HOST; read before the call returns
 *   T_cw_dev     NULL, or a DEVICE float[12] pose that overrides cam->T_cw and is read on the stream (so that a
 *                tracking loop updates the pose on the device without host synchronisation)
 * Writes per-Gaussian features and tile rectangles into the context.  A Gaussian is culled when z_c <= near_z,
 * opacity < 1/255, its projection is non-finite or its extent {alpha >= 1/255} covers no pixel. */
GS_API int gs_preprocess(gs_ctx* ctx, void* stream, int64_t N, int sh_degree, const float* means, const float* scales,
                  const float* quats, const float* opacities, const float* sh, const gs_camera* cam,
                  const float* T_cw_dev);

/* Steps a2-a5 -- per-tile instance lists ordered by (depth key, Gaussian index)  (Q13).  The sort on (tile id, depth
 * bits, index) keys is split MSD-first: counting pass on the tile digit (per-tile counts by gs_preprocess, multi-CTA
 * prefix sum = the per-tile ranges, duplication into tile buckets with an 8-bit mask of the 8x4-pixel regions of the
 * tile the Gaussian can reach), then a register-resident bitonic sort of every bucket on its unique 64-bit keys: the
 * result is THE (tile, depth, index) order, bit for bit (DESIGN.md section 6 records the measured radix alternatives).
 * The first call after gs_create (or after N / the image size changed) synchronises once to size the instance
 * buffers; later calls are asynchronous and report an overflow through GS_E_OVERFLOW on a later call.
 * The prefix-sum kernel exchanges per-CTA totals through {epoch, value} words its CTAs poll: it is launched cooperatively
 * (all of its <= 128 CTAs are guaranteed co-resident; GS_E_CUDA if the device cannot hold them, e.g. under MPS limits).
 * Stream behaviour of the five calls: every kernel is launched on `stream` with the programmatic-stream-serialization
 * attribute and begins with griddepcontrol.wait, i.e. it consumes nothing before the work in front of it on the stream
 * (the caller's own kernels included) has completed; work the caller enqueues behind a call is ordered as usual.  Only
 * buckets beyond 2047 keys are sorted on a context-owned side stream (forked from and joined to `stream` by events), and
 * only in iterations that follow one that had such buckets.
 * Once per gs_preprocess: the scan consumes (and clears) the per-tile counters, a second call returns GS_E_ORDER. */
GS_API int gs_bin_tiles(gs_ctx* ctx, void* stream);

/* Step a6 -- per-tile front-to-back compositing (oracle reading C1 step 7).
 *   bg     HOST float[3] background colour (NULL = black); rgb_out = C + T_final * bg
 *   rgb    [3,H,W]; depth [H,W] = sum z_c alpha T (un-normalised, Q8); alpha [H,W] = 1 - T_final.  Any may be NULL. */
GS_API int gs_rasterize_fwd(gs_ctx* ctx, void* stream, const float* bg, float* rgb, float* depth, float* alpha);

/* Steps a8-a9 -- back-to-front per-pixel backward (per-Gaussian sums reduced over the 32 pixels of a warp's region
 * through shared memory, then one coalesced set of global RED.ADD per (region, Gaussian) into per-Gaussian 2-D
 * gradients), then the per-Gaussian chain rule (oracle readings C2, C3).
 *   d_rgb [3,H,W], d_depth [H,W] (NULL = 0), d_alpha [H,W] (NULL = 0): upstream gradients of the three outputs
 *   flags: GS_ACCUMULATE, GS_POSE_ONLY
 *   g_means [N,3], g_scales [N,3], g_quats [N,4], g_opacities [N], g_sh [N,K,3]: gradients w.r.t. the ABI parameters
 *   (activated scales / opacities, raw quaternions, SH coefficients); exact zeros for culled Gaussians.  With
 *   GS_POSE_ONLY they are not touched and may be NULL. */
GS_API int gs_rasterize_bwd(gs_ctx* ctx, void* stream, const float* d_rgb, const float* d_depth, const float* d_alpha,
                     uint32_t flags, float* g_means, float* g_scales, float* g_quats, float* g_opacities, float* g_sh);

/* Step a10 -- 6-DoF pose gradient (oracle reading C4): dL/dxi at xi = 0 for T_cw <- Exp(xi^) T_cw, xi = (rho, phi).
 *   g_twist  DEVICE float[6]: rho_x, rho_y, rho_z, phi_x, phi_y, phi_z (overwritten, or added to with GS_ACCUMULATE).
 * Must follow gs_rasterize_bwd of the same iteration. */
GS_API int gs_pose_grad(gs_ctx* ctx, void* stream, uint32_t flags, float* g_twist);

/* ---- introspection (tests, benchmarks) ------------------------------------------------------------------------ */
/* Number of visible Gaussians and of tile instances of the last gs_bin_tiles.  SYNCHRONISES the stream. */
GS_API int gs_get_counts(gs_ctx* ctx, void* stream, int64_t* n_visible, int64_t* n_instances);
/* Sorted keys [I] (tile << 32 | depth bits), sorted Gaussian ids [I], tile ranges [tiles,2] = [begin,end). */
GS_API int gs_get_binning(gs_ctx* ctx, void* stream, uint64_t* keys_sorted, uint32_t* ids_sorted, uint32_t* tile_ranges);
/* Per-Gaussian features of the last gs_preprocess.  mean2d double[N,2] (integer + fraction, exact), conic float[N,3]
 * (a,b,c of Sigma'^-1), color float[N,3], depth float[N] (z_c), depth_key uint32[N] (bits of the canonical fp32
 * depth), rect int32[N,4] tile rectangle tx0,ty0,tx1,ty1 (half-open; all zero = culled).  Any may be NULL. */
GS_API int gs_get_features(gs_ctx* ctx, void* stream, double* mean2d, float* conic, float* color, float* depth,
                    uint32_t* depth_key, int32_t* rect);
/* DEVICE pointers (context-owned, valid until the next gs_preprocess) to the compacted indices of the visible Gaussians of
 * the last gs_preprocess, uint32[n_visible] in visible-slot order (arbitrary but fixed for the iteration), and to the count
 * itself: the row order of GS_SPARSE_GRADS gradients.  No synchronisation. */
GS_API int gs_visible_ids(gs_ctx* ctx, const uint32_t** ids, const uint32_t** n_visible);
/* Copies that index list into caller-owned DEVICE memory ids_out uint32[N] (entries beyond n_visible are unspecified);
 * asynchronous on `stream`. */
GS_API int gs_get_visible_ids(gs_ctx* ctx, void* stream, uint32_t* ids_out);
/* Non-blocking: GS_E_OVERFLOW if an earlier asynchronous iteration overflowed the instance capacity, else GS_OK.  Covers
 * the context and the view sub-contexts of gs_refine_views (GS_OPT_VIEW_STREAMS > 1): a view that overflowed on any of
 * them is reported here after the stream has been synchronised, and at the entry of the next gs_refine_views. */
GS_API int gs_poll(gs_ctx* ctx);

/* Stage timing.  gs_profile_enable(ctx, 1) makes the five calls record CUDA events on their stream around each kernel
 * group; gs_profile_read waits for the last gs_pose_grad and returns the device time in milliseconds of the
 * GS_NUM_STAGES groups of the last iteration: preprocess, tile scan, duplication (emit), per-tile sort, raster forward,
 * raster backward (pixel part), per-Gaussian backward, pose gradient.  HOST float[GS_NUM_STAGES]. */
#define GS_NUM_STAGES 8
GS_API int gs_profile_enable(gs_ctx* ctx, int on);
GS_API int gs_profile_read(gs_ctx* ctx, float* ms);
/* Number of CUDA kernels this context has launched so far (HOST counter). */
GS_API int gs_get_launch_count(gs_ctx* ctx, uint64_t* n);
/* Workload of the last forward (SYNCHRONISES; re-walks the lists with the forward's own decisions): HOST
 * uint64[GS_NUM_WORKLOAD] = { E: (pixel, Gaussian) pairs evaluated while the pixel was still alive, over the (region,
 * Gaussian) entries the region masks keep; C: blended pairs; L: sum over pixels of the last blended list position;
 * sum over pixels of their tile's list length; R: relevant (8x4 region, Gaussian) entries walked by the forward;
 * Eb: pairs the backward must evaluate (relevant entries up to each pixel's last blended one); Rb: relevant entries the
 * backward walks (up to each region's last blended one) }. */
#define GS_NUM_WORKLOAD 7
GS_API int gs_get_workload(gs_ctx* ctx, void* stream, uint64_t* out);

/* ---- auxiliary kernels outside the five-call contract (losses of configs 2 and 4, on-device pose step) ---------- */
/* grad[i] = weight * sign(pred[i] - target[i])   (d/dpred of weight * |pred - target|; sign(0) = 0) */
GS_API int gs_aux_l1_grad(void* stream, int64_t n, const float* pred, const float* target, float weight, float* grad);
/* T_cw <- Exp(-step * g / |g|) T_cw on the device (normalised gradient step; no-op if |g| = 0).  T_cw_dev float[12]. */
GS_API int gs_aux_pose_step(void* stream, float* T_cw_dev, const float* g_twist, float step);

/* ---- mapping-loss terms of Eq. 4 that need no dataset ---------------------------------------- */
/* alpha L1(I^, I) + beta L1(D^, D) (paper: alpha = 0.95, beta = 0.25).  Reading (Q18): L1(I^, I) = mean over the
 * 3 H W values of |I^ - I|; L1(D^, D) = (1 / H W) sum over pixels with target_depth > 0 of |D^ - D|; sign(0) = 0.
 * Inputs: DEVICE float rgb, target_rgb [3,H,W]; depth, target_depth [H,W].  Outputs: DEVICE d_rgb [3,H,W] =
 * alpha sign(I^ - I) / (3 H W), d_depth [H,W] = beta sign(D^ - D) / (H W) (0 where target_depth <= 0) -- directly the
 * upstream gradients of gs_rasterize_bwd -- and DEVICE double loss[4] = { L1 rgb, L1 depth, alpha L1 rgb + beta L1 depth,
 * scratch }.
 * Asynchronous on `stream`; all arrays caller-owned.  GS_E_INVALID on a null pointer or an empty image. */
GS_API int gs_loss_map(void* stream, int32_t width, int32_t height, const float* rgb, const float* depth,
                       const float* target_rgb, const float* target_depth, float alpha, float beta, float* d_rgb,
                       float* d_depth, double* loss);
/* lambda_s L_iso = lambda_s sum_i |s_i - mean(s_i)|_1 over the three (activated) scale components (paper: lambda_s =
 * 10).  DEVICE scales [N,3]; its gradient is ADDED into DEVICE g_scales [N,3] (call after gs_rasterize_bwd);
 * DEVICE double loss[2]: loss[0] = the weighted loss (loss[1] is scratch). */
GS_API int gs_loss_iso(void* stream, int64_t N, const float* scales, float lambda_s, float* g_scales, double* loss);

/* ---- refinement loss of the fused map, Eq. 23, without its normal term (gs_loss_normal) ---------- */
/* On the exposure-compensated render I~ = e^a I^ + b (per-keyframe log-gain a and bias b):
 *     L = alpha' L1(I~, I) + lambda (1 - SSIM(I~, I)) + beta L1(D^, D-)       (paper: alpha' = 1.75, lambda = 0.2, beta = 0.25).
 * Readings: Q19 SSIM = 11 x 11 Gaussian window of sigma 1.5, C1 = 0.01^2, C2 = 0.03^2, zero padding, per channel,
 * mean over pixels and channels; Q18 mean reductions, depth term where target_depth > 0, sign(0) = 0.
 * Inputs DEVICE: rgb, target_rgb [3,H,W]; depth, target_depth [H,W]; ab float[2] = (a, b).  Outputs DEVICE: d_rgb [3,H,W] =
 * dL/dI^ and d_depth [H,W] = dL/dD^ (directly the upstream gradients of gs_rasterize_bwd); g_ab float[2] = (dL/da, dL/db);
 * loss double[8] = { L1(I~,I), SSIM(I~,I), L1(D^,D-), L, dL/da, dL/db, scratch, scratch }.  work: DEVICE scratch of 9 H W floats.
 * Asynchronous on `stream` (three launches); all arrays caller-owned.  GS_E_INVALID on a null pointer or an empty image. */
GS_API int gs_loss_refine(void* stream, int32_t width, int32_t height, const float* rgb, const float* depth,
                          const float* target_rgb, const float* target_depth, const float* ab, float alpha_p, float lambda,
                          float beta, float* d_rgb, float* d_depth, float* g_ab, float* work, double* loss);

/* ---- depth-induced normals and the normal term of Eqs. 4 / 23 -------------------------------- */
/* N^ = depth-induced normal of the rendered depth (reading Q22: pinhole back-projection, forward differences,
 * N^ = (t_y x t_x) / |.|, facing the camera; defined off the last column / row where the three depths are > 0), and
 * lambda_n L_normal, L_normal = (1 / H W) sum |1 - N^ . N-| over pixels that have a normal and a non-zero prior N-.
 *   depth         DEVICE [H,W]   rendered depth (gs_rasterize_fwd)
 *   normal_prior  DEVICE [3,H,W] unit normals in camera coordinates, zero vector = no prior; NULL = normals only
 *   normals_out   DEVICE [3,H,W] or NULL: the depth-induced normal map (zeros where undefined)
 *   d_depth       DEVICE [H,W]: lambda_n dL_normal/dD^ is ADDED (call after gs_loss_map / gs_loss_refine wrote it)
 *   loss          DEVICE double[2]: loss[0] = lambda_n L_normal (loss[1] scratch)
 * Asynchronous on `stream`.  GS_E_INVALID on null / inconsistent pointers or an empty image. */
GS_API int gs_loss_normal(void* stream, int32_t width, int32_t height, float fx, float fy, float cx, float cy,
                          const float* depth, const float* normal_prior, float lambda_n, float* normals_out, float* d_depth,
                          double* loss);

/* ---- Eq. 19: a submap's Sim(3) correction applied to its Gaussians --------------------------------- */
/* mu' = s R mu + t, s_i' = s s_i, q' = q_R (x) q (so that Sigma' = s^2 R Sigma R^T); opacity and colour are unchanged
 * and are not arguments.  s > 0, R row-major float[9] (a rotation), t float[3]: HOST.  means, scales
 * [N,3], quats [N,4] (16-byte aligned) and the three outputs: DEVICE; an output may alias its input (in place).
 * Asynchronous on `stream`.  GS_E_INVALID on null pointers, s <= 0 or misaligned quaternions. */
GS_API int gs_sim3_apply(void* stream, int64_t N, float s, const float* R, const float* t, const float* means,
                         const float* scales, const float* quats, float* means_out, float* scales_out, float* quats_out);

/* ---- Eqs. 20-22: occupancy-aware fusion ---------------------------------------------------- */
/* Voxel sets are open-addressing hash tables of 64-bit spatial-hash keys in CALLER-provided DEVICE memory: uint64
 * table[capacity], capacity a power of two, empty slot = 0xFFFFFFFFFFFFFFFF.  Readings (Q21): kappa(x) = floor(x / v)
 * per axis (fp64), key = (ix + 2^20) | (iy + 2^20) << 21 | (iz + 2^20) << 42; the box of Eq. 20 is axis-aligned in world
 * coordinates with half extents k s_i; r_k(u) = back-projection of integer-centred pixel u at its camera-space depth; pixels
 * with depth <= 0 cast no ray; the voxels of a ray are those of the 3-D DDA in fp64 (bit-identical to the plain definition
 * of Eq. 21).  v (voxel) and k are unpublished: arguments.  `overflow` (DEVICE uint32, caller-zeroed) counts keys that
 * could not be stored (table full, index beyond 21 bits, non-finite input): the sets are exact iff it stays 0.
 * "Table full" means: no free slot within 128 probes of the key's home slot (size the tables for a load factor <= 0.5);
 * a Gaussian whose box of Eq. 20 covers more than 2^24 voxels is not inserted and counted once, and a ray or a large box
 * is given up at its first key that finds no room (the count is of failed attempts: zero or non-zero is what it tells) -- an undersized
 * table or a runaway scale ends in a prompt overflow report, never in a long-running kernel.  gs_voxel_retain never retains a Gaussian with a non-finite mean.
 * All calls are asynchronous on `stream`; GS_E_INVALID on null pointers, non-power-of-two capacities, voxel <= 0. */
GS_API int gs_voxel_set_clear(void* stream, uint64_t* table, int64_t capacity);
/* O_occ (Eq. 20) of target Gaussians: DEVICE means, scales [N,3] (activated scales). */
GS_API int gs_voxel_insert_boxes(void* stream, uint64_t* table, int64_t capacity, float voxel, float k, int64_t N,
                                 const float* means, const float* scales, uint32_t* overflow);
/* O_free (Eq. 21) of one keyframe: cam HOST (intrinsics, world-to-camera pose), DEVICE depth [H,W]; every `stride`-th pixel
 * in x and y casts a ray (stride 1 = every pixel, as in the paper). */
GS_API int gs_voxel_insert_rays(void* stream, uint64_t* table, int64_t capacity, float voxel, const gs_camera* cam,
                                const float* depth, int32_t stride, uint32_t* overflow);
/* Eq. 22: retain[j] = 1 iff kappa(mu_j) is in neither set (either table may be NULL = empty set).  DEVICE uint8 retain[N]. */
GS_API int gs_voxel_retain(void* stream, const uint64_t* occ, int64_t occ_capacity, const uint64_t* free_set,
                           int64_t free_capacity, float voxel, int64_t N, const float* means, uint8_t* retain);

/* ---- optimiser step and pruning of the refinement ------------------------------------------------ */
/* The five parameter arrays of a Gaussian set (DEVICE pointers; shapes as in gs_preprocess: [N,3], [N,3], [N,4], [N], [N,K,3]). */
typedef struct { float* means; float* scales; float* quats; float* opacities; float* sh; } gs_gaussians;
typedef struct {
  float lr_means, lr_scales, lr_quats, lr_opacities, lr_sh; /* learning rate per parameter group */
  float beta1, beta2, eps;                                  /* Adam constants (0.9, 0.999, 1e-15) */
  int32_t step;                                             /* 1-based iteration number t of the bias correction */
} gs_adam_config;
/* One fused Adam step (reading Q20: the paper says only "gradient descent" and "learning rate"): Kingma & Ba
 * Algorithm 1 with bias correction; centres, raw quaternions and SH directly, scales through log s and opacities through
 * logit o, so the ACTIVATED values of this ABI stay in (0, inf) / (0, 1).  grads = gradients w.r.t. the activated values
 * (the outputs of gs_rasterize_bwd); m, v = first / second moments, same shapes as the parameters, caller-zeroed at start.
 * visible: NULL, or DEVICE uint32[N]: only Gaussians with a non-zero entry are touched (parameters and moments).
 * cfg HOST.  In place, asynchronous (five launches).  GS_E_INVALID on null pointers, degree outside 0..3, step < 1. */
GS_API int gs_adam_step(void* stream, int64_t N, int sh_degree, const gs_adam_config* cfg, const gs_gaussians* params,
                        const gs_gaussians* grads, const gs_gaussians* m, const gs_gaussians* v, const uint32_t* visible);
/* The same step on GS_SPARSE_GRADS gradients: grads arrays hold one row per visible Gaussian, row r -> Gaussian ids[r],
 * r < *n_rows (DEVICE count, e.g. from gs_visible_ids); max_rows >= *n_rows bounds the launch (N is always enough).
 * Touches exactly the Gaussians listed (parameters and moments), like gs_adam_step with a visibility mask. */
GS_API int gs_adam_step_sparse(void* stream, int64_t N, int sh_degree, const gs_adam_config* cfg, const gs_gaussians* params,
                               const gs_gaussians* grads, const gs_gaussians* m, const gs_gaussians* v, const uint32_t* ids,
                               const uint32_t* n_rows, int64_t max_rows);
/* keep[i] = opacities[i] >= min_opacity  ("prunes Gaussians with opacity below 0.005").  DEVICE uint8 keep[N]. */
GS_API int gs_prune_mask(void* stream, int64_t N, const float* opacities, float min_opacity, uint8_t* keep);
/* Order-preserving stream compaction, shared by pruning and by the retain test of Eq. 22.  gs_compact_plan turns a keep
 * mask into index[i] = destination row of Gaussian i (0xFFFFFFFF if dropped) and the DEVICE count n_kept; work = DEVICE
 * scratch of gs_compact_work_bytes(N) bytes.  gs_compact_rows gathers the kept rows of one [N,width] float array into
 * `out` (must not alias `in`; rows beyond n_kept are untouched).  N < 2^32. */
GS_API int64_t gs_compact_work_bytes(int64_t N);
GS_API int gs_compact_plan(void* stream, int64_t N, const uint8_t* keep, uint32_t* index, int64_t* n_kept, void* work);
GS_API int gs_compact_rows(void* stream, int64_t N, int32_t width, const uint32_t* index, const float* in, float* out);
/* gs_compact_plan for callers that must not allocate device memory where they compact.  Two kinds of caller are meant:
 * a long-running agent that sized all of its device buffers at start-up and handed the rest of HBM to its own pool, so a
 * cudaMalloc in the middle of a mission can fail (or fragment the pool it does not know about); and a loop that prunes or
 * fuses (Eq. 22) while tracking and mapping kernels run on other streams, where cudaMalloc / cudaFree would
 * stall all of them, because both synchronise the whole device.  Such callers already own keep / index / n_kept; the one
 * thing gs_compact_plan still asks them to find room for is its scratch.  Here that scratch is a fixed array inside the
 * library image (64 KiB, one uint32 per 1024 Gaussians): every GPU that loads libgs.so holds it until the process exits.
 *   - Same arguments (minus `work`), same outputs, bit for bit, as gs_compact_plan.  Asynchronous on `stream`, which must
 *     belong to the CURRENT device (the scratch used is the current device's copy).
 *   - Limit: N <= gs_compact_plan_static_max() = 16 777 216 Gaussians.  A larger N returns GS_E_TOO_LARGE and launches
 *     nothing; use gs_compact_plan with caller scratch for such maps.
 *   - The call never calls cudaMalloc, cudaFree or any routine that allocates.  The FIRST call on each device looks up
 *     the array's device address (cudaGetSymbolAddress, once per device, mutex-guarded); make that first call during
 *     set-up, before any stream capture; a call with N = 0 (it only clears *n_kept) is enough.
 *   - All calls on one device share the one array and it keeps whatever the last call left.  That is harmless for calls
 *     that follow one another on a stream (every word read is written earlier in the same call; nothing needs zeroing),
 *     but two calls whose kernels can overlap on the GPU (different streams, no dependency between them) RACE on it and
 *     both results are garbage.  Order them with an event, or give one of them gs_compact_plan with its own scratch. */
GS_API int64_t gs_compact_plan_static_max(void);
GS_API int gs_compact_plan_static(void* stream, int64_t N, const uint8_t* keep, uint32_t* index, int64_t* n_kept);

/* ---- one whole iteration of the joint refinement (Eq. 23) over a batch of keyframe views ----------- */
/* For every view k: gs_preprocess -> gs_bin_tiles -> gs_rasterize_fwd -> gs_loss_refine on I~ = e^{a_k} I^ + b_k (+ gs_loss_normal
 * if normal priors are given) -> gs_rasterize_bwd with the parameter gradients ACCUMULATED over the views -> gs_pose_grad:
 * everything the refinement differentiates (the fused Gaussians, the per-keyframe pose deltas and the per-keyframe log-gain
 * and bias) in one call, no framework op and no host synchronisation in between.  All views share one image size.
 *   batch (HOST struct): cams HOST [n_views]; T_cw_dev NULL or DEVICE [n_views,12] poses that override the cams' (pose
 *     deltas applied on the device); target_rgb DEVICE [n_views,3,H,W]; target_depth DEVICE [n_views,H,W]; normal_prior NULL
 *     or DEVICE [n_views,3,H,W]; ab DEVICE [n_views,2]; the weights of Eq. 23 (paper: 1.75, 0.2, 0.25; lambda_n garbled, Q16).
 *   grads      DEVICE arrays of the parameter shapes: sum over the views of dL_k/dparam (written by view 0, accumulated after;
 *              with GS_OPT_VIEW_STREAMS > 1: zeroed first, accumulated by all views in whatever order they finish)
 *   g_twist    DEVICE [n_views,6]; g_ab DEVICE [n_views,2]
 *   loss       DEVICE double [n_views,10]: the eight entries of gs_loss_refine, then lambda_n L_normal and a scratch word
 *   visible    NULL or DEVICE uint32[N]: 1 where the Gaussian was on screen in at least one view (the mask of gs_adam_step)
 * The rendered images live in context-owned scratch.  Same asynchrony and overflow protocol as the five calls. */
typedef struct {
  int32_t n_views;
  const gs_camera* cams;
  const float* T_cw_dev;
  const float* target_rgb;
  const float* target_depth;
  const float* normal_prior;
  const float* ab;
  float alpha_p, lambda, beta, lambda_n;
} gs_refine_batch;
GS_API int gs_refine_views(gs_ctx* ctx, void* stream, int64_t N, int sh_degree, const gs_gaussians* params,
                           const gs_refine_batch* batch, const float* bg, const gs_gaussians* grads, float* g_twist, float* g_ab,
                           double* loss, uint32_t* visible);

/* ---- measured machine peaks: the denominators of bench.py's roofline entries -------- */
/* Runs small synthetic kernels on `device` (allocates and frees ~2 GiB, synchronises; ~0.2 s) and fills HOST double
 * out[GS_NUM_PEAKS]:  FP32 FMA lane rate (T lane-FMA/s; x2 = TFLOP/s), mixed FFMA+integer issue rate (T warp
 * instructions/s), MUFU.EX2 rate (T lanes/s), shared-memory load rates in T warp-level LDS/s (128-bit broadcast = how the
 * compositing kernels read a Gaussian record; 128-bit conflict-free; 32- and 64-bit broadcast), L2 RED.ADD.F32 rate
 * (G lane-adds/s on 128-byte rows), HBM read / write / copy (GB/s, 1 GiB streams), SM count and maximum SM clock (MHz).
 * None of the method's arithmetic is involved.  GS_E_NOMEM if the buffers cannot be allocated. */
#define GS_PEAK_FMA_TLANES 0
#define GS_PEAK_ISSUE_TWARP 1
#define GS_PEAK_EX2_TLANES 2
#define GS_PEAK_LDS128_BCAST_TWARP 3
#define GS_PEAK_LDS128_TWARP 4
#define GS_PEAK_LDS32_BCAST_TWARP 5
#define GS_PEAK_LDS64_BCAST_TWARP 6
#define GS_PEAK_RED_GLANES 7
#define GS_PEAK_HBM_READ_GBS 8
#define GS_PEAK_HBM_WRITE_GBS 9
#define GS_PEAK_HBM_COPY_GBS 10
#define GS_PEAK_SM_COUNT 11
#define GS_PEAK_SM_MHZ_MAX 12
#define GS_NUM_PEAKS 13
GS_API int gs_measure_peaks(int device, void* stream, double* out);

/* ---- host-buffer convenience (bench.py "e2e"): one whole fwd+bwd iteration with HOST arrays -------------------- */
/* Copies the parameters host->device, runs the five steps with the given upstream gradients (HOST), copies the image
 * and all gradients device->host and synchronises.  Pointers follow the shapes above; outputs may be NULL. */
GS_API int gs_fwd_bwd_host(gs_ctx* ctx, void* stream, int64_t N, int sh_degree, const float* means, const float* scales,
                    const float* quats, const float* opacities, const float* sh, const gs_camera* cam, const float* bg,
                    const float* d_rgb, const float* d_depth, float* rgb, float* depth, float* alpha, float* g_means,
                    float* g_scales, float* g_quats, float* g_opacities, float* g_sh, float* g_twist);
/* The same without the final synchronisation: everything is enqueued on `stream` and the call returns.  The host arrays
 * must be page-locked and must not be touched until the caller has synchronised the stream (then gs_poll reports an
 * overflow of that iteration).  Two contexts on two streams fed alternately overlap one iteration's device->host copies
 * with the next one's host->device copies and kernels (PCIe is full duplex): bench.py "e2e". */
GS_API int gs_fwd_bwd_host_async(gs_ctx* ctx, void* stream, int64_t N, int sh_degree, const float* means,
                          const float* scales, const float* quats, const float* opacities, const float* sh,
                          const gs_camera* cam, const float* bg, const float* d_rgb, const float* d_depth, float* rgb,
                          float* depth, float* alpha, float* g_means, float* g_scales, float* g_quats, float* g_opacities,
                          float* g_sh, float* g_twist);

#ifdef __cplusplus
}
#endif
#endif /* GS_H_ */

// gs_api.cu -- the extern "C" boundary of libgs.so (include/gs.h): context, scratch, call sequencing, introspection,
// auxiliary kernels and the host-buffer convenience path.  Argument marshalling and launches only.
#include <math.h>
#include <new>
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "gs_internal.cuh"

using namespace gs;

namespace gs {

__global__ void features_export_kernel(int64_t N, const float4* __restrict__ feat, const uint4* __restrict__ vis_rec,
                                       const uint32_t* __restrict__ tiles_touched,
                                       const uint32_t* __restrict__ slot_of, double* mean2d, float* conic,
                                       float* color, float* depth, uint32_t* dkey, int32_t* rect_out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const bool vis = tiles_touched[i] > 0;
  float4 f0 = make_float4(0, 0, 0, 0), f1 = f0, f2 = f0;
  ushort4 r = make_ushort4(0, 0, 0, 0);
  uint32_t dk = 0;
  if (vis) {
    const size_t k = slot_of[i];  // the feature records are stored by visible slot
    f0 = feat[3 * k]; f1 = feat[3 * k + 1]; f2 = feat[3 * k + 2];
    const uint4 rec = vis_rec[k];  // {tx0 | ty0 << 16, tx1 | ty1 << 16, depth key, index}
    r = make_ushort4((unsigned short)(rec.x & 0xffffu), (unsigned short)(rec.x >> 16), (unsigned short)(rec.y & 0xffffu),
                     (unsigned short)(rec.y >> 16));
    dk = rec.z;
  }
  const double ln2 = 0.6931471805599453;
  if (mean2d) {
    const int pk = __float_as_int(f0.z);
    mean2d[2 * i] = vis ? (double)((pk << 16) >> 16) + (double)f0.x : 0.0;
    mean2d[2 * i + 1] = vis ? (double)(pk >> 16) + (double)f0.y : 0.0;
  }
  if (conic) {  // 0.5 log2(e) Q = L L^T  (gs_internal.cuh)
    const double l11 = f1.x, l21 = f1.y, l22 = f1.z;
    conic[3 * i] = (float)(2.0 * ln2 * l11 * l11);
    conic[3 * i + 1] = (float)(2.0 * ln2 * l11 * l21);
    conic[3 * i + 2] = (float)(2.0 * ln2 * (l21 * l21 + l22 * l22));
  }
  if (color) { color[3 * i] = f2.x; color[3 * i + 1] = f2.y; color[3 * i + 2] = f2.z; }
  if (depth) depth[i] = f2.w;
  if (dkey) dkey[i] = dk;
  if (rect_out) { rect_out[4 * i] = r.x; rect_out[4 * i + 1] = r.y; rect_out[4 * i + 2] = r.z; rect_out[4 * i + 3] = r.w; }
}

__global__ void l1_grad_kernel(int64_t n, const float* __restrict__ pred, const float* __restrict__ target, float weight,
                               float* __restrict__ grad) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float d = pred[i] - target[i];
  grad[i] = d > 0.f ? weight : (d < 0.f ? -weight : 0.f);
}

// T <- Exp(xi^) T with xi = -step * g / |g|  (fp64, one thread)
__global__ void pose_step_kernel(float* T, const float* __restrict__ g, float step) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double gn = 0.0;
  for (int k = 0; k < 6; ++k) gn += (double)g[k] * g[k];
  gn = sqrt(gn);
  if (!(gn > 0.0) || !isfinite(gn)) return;
  double xi[6];
  for (int k = 0; k < 6; ++k) xi[k] = -(double)step * g[k] / gn;
  const double* rho = xi; const double* phi = xi + 3;
  const double th2 = phi[0] * phi[0] + phi[1] * phi[1] + phi[2] * phi[2], th = sqrt(th2);
  double A, B, C;
  if (th < 1e-6) { A = 1.0 - th2 / 6.0; B = 0.5 - th2 / 24.0; C = 1.0 / 6.0 - th2 / 120.0; }
  else { A = sin(th) / th; B = (1.0 - cos(th)) / th2; C = (th - sin(th)) / (th2 * th); }
  const double Kx[9] = {0, -phi[2], phi[1], phi[2], 0, -phi[0], -phi[1], phi[0], 0};
  double K2[9], R[9], V[9];
  for (int r = 0; r < 3; ++r)
    for (int c = 0; c < 3; ++c) K2[3 * r + c] = Kx[3 * r] * Kx[c] + Kx[3 * r + 1] * Kx[3 + c] + Kx[3 * r + 2] * Kx[6 + c];
  for (int k = 0; k < 9; ++k) {
    const double I = (k % 4 == 0) ? 1.0 : 0.0;
    R[k] = I + A * Kx[k] + B * K2[k];
    V[k] = I + B * Kx[k] + C * K2[k];
  }
  double Told[12], Tn[12];
  for (int k = 0; k < 12; ++k) Told[k] = T[k];
  for (int r = 0; r < 3; ++r) {
    for (int c = 0; c < 3; ++c) Tn[4 * r + c] = R[3 * r] * Told[c] + R[3 * r + 1] * Told[4 + c] + R[3 * r + 2] * Told[8 + c];
    Tn[4 * r + 3] = R[3 * r] * Told[3] + R[3 * r + 1] * Told[7] + R[3 * r + 2] * Told[11] + V[3 * r] * rho[0] +
                    V[3 * r + 1] * rho[1] + V[3 * r + 2] * rho[2];
  }
  for (int k = 0; k < 12; ++k) T[k] = (float)Tn[k];
}

static int ensure_gaussian_capacity(gs_ctx* ctx, int64_t N) {
  if (N <= ctx->cap_N) return GS_OK;
  GS_CUDA(cudaDeviceSynchronize());
  const int64_t cap = N + N / 8 + 1024;
  int rc;
  if ((rc = grow(ctx, ctx->feat, 3 * cap)) != GS_OK) return rc;
  if ((rc = grow(ctx, ctx->tiles_touched, cap + 4)) != GS_OK) return rc;
  if ((rc = grow(ctx, ctx->vis_ids, cap)) != GS_OK) return rc;
  if ((rc = grow(ctx, ctx->vis_rec, cap)) != GS_OK) return rc;
  if ((rc = grow(ctx, ctx->vis_par, 3 * cap)) != GS_OK) return rc;
  if ((rc = grow(ctx, ctx->slot_of, cap)) != GS_OK) return rc;
  if ((rc = grow(ctx, ctx->g2d, cap * kG2D)) != GS_OK) return rc;
  GS_CUDA(cudaMemset(ctx->g2d, 0, (size_t)cap * kG2D * sizeof(float)));
  ctx->g2d_dirty = false;
  ctx->cap_N = cap;
  return GS_OK;
}

// One allocation holds everything gs_preprocess must zero at the start of an iteration, so that it is ONE memset:
// [Counts, 128 B][pose accumulators, 16 doubles][per-tile instance counters, one per 128-byte line].
static int alloc_header(gs_ctx* ctx, int64_t tiles) {
  if (ctx->hdr) cudaFree(ctx->hdr);
  ctx->hdr = nullptr;
  const size_t bytes = kHdrBytes + (size_t)tiles * kCtrStride * sizeof(uint32_t);
  if (cudaMalloc((void**)&ctx->hdr, bytes) != cudaSuccess || cudaMemset(ctx->hdr, 0, bytes) != cudaSuccess) {
    cudaGetLastError();
    ctx->hdr = nullptr;
    return fail(ctx, GS_E_NOMEM, "cudaMalloc failed while growing scratch");
  }
  ctx->counts = reinterpret_cast<Counts*>(ctx->hdr);
  ctx->pose_acc = reinterpret_cast<double*>(ctx->hdr + 128);
  ctx->tile_count = reinterpret_cast<uint32_t*>(ctx->hdr + kHdrBytes);
  ctx->hdr_clean = true;
  ctx->ctr_dirty = 0;
  return GS_OK;
}

// visible[i] = 1 where the Gaussian was on screen in this view (the mask is zeroed before the first view; every writer
// writes the same 1, so views on different streams may run this at the same time)
__global__ void visible_or_kernel(int64_t N, const uint32_t* __restrict__ tiles_touched, uint32_t* __restrict__ visible) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < N && tiles_touched[i] > 0u) visible[i] = 1u;
}

static int ensure_image_capacity(gs_ctx* ctx, int64_t tiles, int64_t pix) {
  int rc;
  if (tiles > ctx->cap_tiles) {
    GS_CUDA(cudaDeviceSynchronize());
    if ((rc = grow(ctx, ctx->ranges, tiles)) != GS_OK) return rc;
    if ((rc = grow(ctx, ctx->tile_order, tiles)) != GS_OK) return rc;
    if ((rc = alloc_header(ctx, tiles)) != GS_OK) return rc;
    if ((rc = grow(ctx, ctx->tile_cursor, tiles * kCtrStride)) != GS_OK) return rc;
    ctx->cap_tiles = tiles;
  }
  if (pix > ctx->cap_pix) {
    GS_CUDA(cudaDeviceSynchronize());
    if ((rc = grow(ctx, ctx->final_T, pix)) != GS_OK) return rc;
    if ((rc = grow(ctx, ctx->n_contrib, pix)) != GS_OK) return rc;
    ctx->cap_pix = pix;
  }
  return GS_OK;
}

}  // namespace gs

extern "C" {

int gs_create(gs_ctx** out, int device) {
  if (!out) return GS_E_INVALID;
  *out = nullptr;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); return GS_E_CUDA; }
  gs_ctx* ctx = new (std::nothrow) gs_ctx();
  if (!ctx) return GS_E_NOMEM;
  ctx->device = device;
  bool ok = cudaSetDevice(device) == cudaSuccess;
  ok = ok && alloc_header(ctx, 0) == GS_OK;
  ok = ok && cudaHostAlloc((void**)&ctx->mailbox, sizeof(Counts), cudaHostAllocMapped) == cudaSuccess;
  // the side stream sorts the few long buckets beside tile_sort_kernel: highest priority, so that its 512-thread CTAs are
  // placed first (launched behind the programmatically pre-launched tile_sort_kernel they otherwise queued until all 3225
  // of its CTAs had been dispatched: the two kernels ran one after the other, config 4: 105 us for 57 || 53)
  int prio_lo = 0, prio_hi = 0;
  ok = ok && cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi) == cudaSuccess;
  ok = ok && cudaStreamCreateWithPriority(&ctx->side_stream, cudaStreamNonBlocking, prio_hi) == cudaSuccess;
  ok = ok && cudaEventCreateWithFlags(&ctx->ev_fork2, cudaEventDisableTiming) == cudaSuccess;
  ok = ok && cudaEventCreateWithFlags(&ctx->ev_join2, cudaEventDisableTiming) == cudaSuccess;
  if (ok) {
    memset(ctx->mailbox, 0, sizeof(Counts));
    ok = cudaHostGetDevicePointer((void**)&ctx->mailbox_dev, ctx->mailbox, 0) == cudaSuccess;
  }
  if (!ok) { cudaGetLastError(); gs_destroy(ctx); return GS_E_CUDA; }
  *out = ctx;
  return GS_OK;
}

int gs_destroy(gs_ctx* ctx) {
  if (!ctx) return GS_E_INVALID;
  cudaSetDevice(ctx->device);
  cudaDeviceSynchronize();
  for (int k = 0; k < 7; ++k) {
    if (ctx->sub[k]) gs_destroy(ctx->sub[k]);
    if (ctx->sub_stream[k]) cudaStreamDestroy(ctx->sub_stream[k]);
    if (ctx->ev_view_join[k]) cudaEventDestroy(ctx->ev_view_join[k]);
  }
  if (ctx->ev_view_fork) cudaEventDestroy(ctx->ev_view_fork);
  cudaFree(ctx->feat); cudaFree(ctx->tiles_touched); cudaFree(ctx->vis_ids); cudaFree(ctx->vis_rec); cudaFree(ctx->vis_par); cudaFree(ctx->slot_of);
  cudaFree(ctx->g2d);
  for (int b = 0; b < 2; ++b) cudaFree(ctx->keys[b]);
  cudaFree(ctx->inst_rec);
  cudaFree(ctx->hdr); cudaFree(ctx->tile_cursor); cudaFree(ctx->scan_ws);
  cudaFree(ctx->ranges); cudaFree(ctx->tile_order); cudaFree(ctx->final_T); cudaFree(ctx->n_contrib);
  cudaFree(ctx->hb); cudaFree(ctx->stats_ws); cudaFree(ctx->rv);
  if (ctx->mailbox) cudaFreeHost(ctx->mailbox);
  if (ctx->side_stream) cudaStreamDestroy(ctx->side_stream);
  if (ctx->ev_fork2) cudaEventDestroy(ctx->ev_fork2);
  if (ctx->ev_join2) cudaEventDestroy(ctx->ev_join2);
  if (ctx->ev_made) for (int k = 0; k < 13; ++k) cudaEventDestroy(ctx->ev[k]);
  cudaGetLastError();
  delete ctx;
  return GS_OK;
}

const char* gs_last_error(const gs_ctx* ctx) { return ctx ? ctx->err : "null context"; }

int gs_visible_ids(gs_ctx* ctx, const uint32_t** ids, const uint32_t** n_visible) {
  if (!ctx || !ids || !n_visible) return GS_E_INVALID;
  if (ctx->stage < 1) return fail(ctx, GS_E_ORDER, "gs_visible_ids before gs_preprocess");
  *ids = ctx->vis_ids;
  *n_visible = &ctx->counts->n_visible;
  return GS_OK;
}

int gs_get_visible_ids(gs_ctx* ctx, void* stream, uint32_t* ids_out) {
  if (!ctx || !ids_out) return GS_E_INVALID;
  if (ctx->stage < 1) return fail(ctx, GS_E_ORDER, "gs_get_visible_ids before gs_preprocess");
  GS_CUDA(cudaSetDevice(ctx->device));
  if (ctx->N > 0)
    GS_CUDA(cudaMemcpyAsync(ids_out, ctx->vis_ids, (size_t)ctx->N * sizeof(uint32_t), cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  return GS_OK;
}

int gs_set_option(gs_ctx* ctx, int option, int value) {
  if (!ctx) return GS_E_INVALID;
  if (option == GS_OPT_EXACT_TILE_CULL) {
    ctx->opt_exact_cull = value != 0;
    for (gs_ctx* c : ctx->sub) if (c) c->opt_exact_cull = value != 0;
    return GS_OK;
  }
  if (option == GS_OPT_VIEW_STREAMS) {
    if (value < 1 || value > 8) return fail(ctx, GS_E_INVALID, "gs_set_option: GS_OPT_VIEW_STREAMS takes 1..8");
    ctx->opt_view_streams = value;
    return GS_OK;
  }
  return fail(ctx, GS_E_INVALID, "gs_set_option: unknown option");
}

// Overflow check of a context AND of the view sub-contexts gs_refine_views runs some of its views on
// (GS_OPT_VIEW_STREAMS > 1): every one that overflowed grows and clears its flag; the first failure is the one reported,
// with the sub-context's message copied into the parent's.
static int handle_overflow_all(gs_ctx* ctx) {
  int rc_all = handle_overflow(ctx);
  for (int k = 0; k < (int)(sizeof(ctx->sub) / sizeof(ctx->sub[0])); ++k) {
    gs_ctx* c = ctx->sub[k];
    if (!c) continue;
    const int rc = handle_overflow(c);
    if (rc != GS_OK && rc_all == GS_OK) {
      rc_all = rc;
      snprintf(ctx->err, sizeof(ctx->err), "view stream %d: %.200s", k + 1, c->err);
    }
  }
  return rc_all;
}

int gs_poll(gs_ctx* ctx) {
  if (!ctx) return GS_E_INVALID;
  return handle_overflow_all(ctx);
}

int gs_preprocess(gs_ctx* ctx, void* stream, int64_t N, int sh_degree, const float* means, const float* scales,
                  const float* quats, const float* opacities, const float* sh, const gs_camera* cam,
                  const float* T_cw_dev) {
  if (!ctx) return GS_E_INVALID;
  if (N < 0 || N >= (1ll << 24) || sh_degree < 0 || sh_degree > 3 || !cam) return fail(ctx, GS_E_INVALID, "gs_preprocess: bad N, sh_degree or camera");
  if (N > 0 && (!means || !scales || !quats || !opacities || !sh)) return fail(ctx, GS_E_INVALID, "gs_preprocess: null parameter array");
  if (cam->width <= 0 || cam->height <= 0 || cam->width > 65535 * GS_TILE || cam->height > 65535 * GS_TILE)
    return fail(ctx, GS_E_INVALID, "gs_preprocess: bad image size");
  if (((uintptr_t)quats & 15) != 0) return fail(ctx, GS_E_INVALID, "gs_preprocess: quats must be 16-byte aligned");
  // the SH rows are read as float4 when a row is a whole number of them (degrees 1 and 3: 12 and 48 floats)
  if ((3 * (sh_degree + 1) * (sh_degree + 1)) % 4 == 0 && ((uintptr_t)sh & 15) != 0)
    return fail(ctx, GS_E_INVALID, "gs_preprocess: sh must be 16-byte aligned for SH degrees 1 and 3");
  cudaStream_t s = (cudaStream_t)stream;
  GS_CUDA(cudaSetDevice(ctx->device));
  int rc;
  if ((rc = handle_overflow(ctx)) != GS_OK) return rc;
  if ((rc = ensure_gaussian_capacity(ctx, N)) != GS_OK) return rc;
  DevCam& c = ctx->cam;
  c.W = cam->width; c.H = cam->height;
  c.tiles_x = (cam->width + GS_TILE - 1) / GS_TILE; c.tiles_y = (cam->height + GS_TILE - 1) / GS_TILE;
  c.fx = cam->fx; c.fy = cam->fy; c.cx = cam->cx; c.cy = cam->cy; c.near_z = cam->near_z;
  memcpy(c.T, cam->T_cw, sizeof(c.T));
  c.T_dev = T_cw_dev;
  if ((rc = ensure_image_capacity(ctx, (int64_t)c.tiles_x * c.tiles_y, (int64_t)c.W * c.H)) != GS_OK) return rc;
  ctx->N = N; ctx->sh_degree = sh_degree;
  ctx->means = means; ctx->scales = scales; ctx->quats = quats; ctx->opacities = opacities; ctx->sh = sh;
  ctx->seq++;
  ctx->counts = reinterpret_cast<Counts*>(ctx->hdr + 64 * (ctx->seq & 1u));
  GS_PROF(0, s);
  // counters, pose accumulators and per-tile instance counters: in the steady state the previous iteration left them
  // zero (gs_internal.cuh kHdrBytes); otherwise (first call, gs_preprocess twice in a row, a calibration pass, N = 0) one memset
  const int64_t tiles_now = (int64_t)c.tiles_x * c.tiles_y;
  if (!ctx->hdr_clean || N == 0 || ctx->ctr_dirty > tiles_now) {
    // (also the counters a LARGER image of an earlier call may have left behind: a scan clears only the tiles it reads)
    GS_CUDA(cudaMemsetAsync(ctx->hdr, 0, kHdrBytes + (size_t)std::max(tiles_now, ctx->ctr_dirty) * kCtrStride * sizeof(uint32_t), s));
    ctx->ctr_dirty = 0;
  }
  ctx->hdr_clean = false;
  ctx->ctr_dirty = std::max(ctx->ctr_dirty, tiles_now);
  ctx->pose_acc_clean = true;
  if ((rc = launch_preprocess(ctx, s)) != GS_OK) return rc;
  GS_PROF(1, s);
  ctx->stage = 1;
  ctx->pose_acc_valid = false;
  return GS_OK;
}

int gs_bin_tiles(gs_ctx* ctx, void* stream) {
  if (!ctx) return GS_E_INVALID;
  if (ctx->stage < 1) return fail(ctx, GS_E_ORDER, "gs_bin_tiles before gs_preprocess");
  // the scan clears the per-tile counters it consumes (no memset in the steady state): a second pass over the same
  // preprocess would read zeros and bin nothing
  if (ctx->stage >= 2) return fail(ctx, GS_E_ORDER, "gs_bin_tiles called twice for one gs_preprocess (its tile counters are consumed)");
  GS_CUDA(cudaSetDevice(ctx->device));
  int rc = launch_binning(ctx, (cudaStream_t)stream);
  if (rc != GS_OK) return rc;
  ctx->stage = 2;
  return GS_OK;
}

int gs_rasterize_fwd(gs_ctx* ctx, void* stream, const float* bg, float* rgb, float* depth, float* alpha) {
  if (!ctx) return GS_E_INVALID;
  if (ctx->stage < 2) return fail(ctx, GS_E_ORDER, "gs_rasterize_fwd before gs_bin_tiles");
  GS_CUDA(cudaSetDevice(ctx->device));
  for (int k = 0; k < 3; ++k) ctx->bg[k] = bg ? bg[k] : 0.f;
  GS_PROF(6, (cudaStream_t)stream);
  int rc = launch_raster_fwd(ctx, (cudaStream_t)stream, rgb, depth, alpha);
  if (rc != GS_OK) return rc;
  GS_PROF(7, (cudaStream_t)stream);
  ctx->stage = 3;
  return GS_OK;
}

int gs_rasterize_bwd(gs_ctx* ctx, void* stream, const float* d_rgb, const float* d_depth, const float* d_alpha,
                     uint32_t flags, float* g_means, float* g_scales, float* g_quats, float* g_opacities, float* g_sh) {
  if (!ctx) return GS_E_INVALID;
  if (ctx->stage < 3) return fail(ctx, GS_E_ORDER, "gs_rasterize_bwd before gs_rasterize_fwd");
  if (!d_rgb) return fail(ctx, GS_E_INVALID, "gs_rasterize_bwd: d_rgb is null");
  const bool write = !(flags & GS_POSE_ONLY);
  if ((flags & GS_SPARSE_GRADS) && (flags & GS_ACCUMULATE))
    return fail(ctx, GS_E_INVALID, "gs_rasterize_bwd: GS_SPARSE_GRADS cannot be combined with GS_ACCUMULATE (the rows of two views differ)");
  if (write && ctx->N > 0 && (!g_means || !g_scales || !g_quats || !g_opacities || !g_sh))
    return fail(ctx, GS_E_INVALID, "gs_rasterize_bwd: null gradient array without GS_POSE_ONLY");
  if (write && ((uintptr_t)g_quats & 15) != 0) return fail(ctx, GS_E_INVALID, "gs_rasterize_bwd: g_quats must be 16-byte aligned");
  if (write && (3 * (ctx->sh_degree + 1) * (ctx->sh_degree + 1)) % 4 == 0 && ((uintptr_t)g_sh & 15) != 0)
    return fail(ctx, GS_E_INVALID, "gs_rasterize_bwd: g_sh must be 16-byte aligned for SH degrees 1 and 3");
  cudaStream_t s = (cudaStream_t)stream;
  GS_CUDA(cudaSetDevice(ctx->device));
  if (ctx->g2d_dirty && ctx->N > 0) GS_CUDA(cudaMemsetAsync(ctx->g2d, 0, (size_t)ctx->N * kG2D * sizeof(float), s));
  ctx->g2d_dirty = true;
  ctx->pose_acc_valid = false;
  GS_PROF(8, s);
  int rc = launch_raster_bwd(ctx, s, d_rgb, d_depth, d_alpha);
  if (rc != GS_OK) return rc;
  GS_PROF(9, s);
  if (write) {
    if ((rc = launch_gauss_bwd(ctx, s, flags, g_means, g_scales, g_quats, g_opacities, g_sh)) != GS_OK) return rc;
  }
  GS_PROF(10, s);
  ctx->stage = 4;
  return GS_OK;
}

int gs_pose_grad(gs_ctx* ctx, void* stream, uint32_t flags, float* g_twist) {
  if (!ctx) return GS_E_INVALID;
  if (ctx->stage < 4) return fail(ctx, GS_E_ORDER, "gs_pose_grad before gs_rasterize_bwd");
  if (!g_twist) return fail(ctx, GS_E_INVALID, "gs_pose_grad: g_twist is null");
  cudaStream_t s = (cudaStream_t)stream;
  GS_CUDA(cudaSetDevice(ctx->device));
  int rc;
  GS_PROF(11, s);
  if (!ctx->pose_acc_valid) {
    if ((rc = launch_gauss_bwd(ctx, s, GS_POSE_ONLY, nullptr, nullptr, nullptr, nullptr, nullptr)) != GS_OK) return rc;
  }
  rc = launch_pose_final(ctx, s, flags, g_twist);
  GS_PROF(12, s);
  return rc;
}

int gs_get_counts(gs_ctx* ctx, void* stream, int64_t* n_visible, int64_t* n_instances) {
  if (!ctx) return GS_E_INVALID;
  if (ctx->stage < 2) return fail(ctx, GS_E_ORDER, "gs_get_counts before gs_bin_tiles");
  GS_CUDA(cudaSetDevice(ctx->device));
  Counts c;
  GS_CUDA(cudaMemcpyAsync(&c, ctx->counts, sizeof(Counts), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  GS_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
  if (n_visible) *n_visible = c.n_visible;
  if (n_instances) *n_instances = c.n_instances;
  if (c.overflow) {
    const int rc = handle_overflow(ctx);
    return rc != GS_OK ? rc : fail(ctx, GS_E_OVERFLOW, "tile-instance capacity exceeded in this iteration; scratch has grown, re-issue");
  }
  return GS_OK;
}

int gs_get_binning(gs_ctx* ctx, void* stream, uint64_t* keys_sorted, uint32_t* ids_sorted, uint32_t* tile_ranges) {
  if (!ctx) return GS_E_INVALID;
  if (ctx->stage < 2) return fail(ctx, GS_E_ORDER, "gs_get_binning before gs_bin_tiles");
  cudaStream_t s = (cudaStream_t)stream;
  GS_CUDA(cudaSetDevice(ctx->device));
  int64_t I = 0;
  int rc = gs_get_counts(ctx, stream, nullptr, &I);
  if (rc != GS_OK) return rc;
  if (keys_sorted && I) {
    if ((rc = export_sorted_keys(ctx, s, keys_sorted)) != GS_OK) return rc;
  }
  if (ids_sorted && I) {
    if ((rc = export_sorted_ids(ctx, s, I, ids_sorted)) != GS_OK) return rc;
  }
  if (tile_ranges)
    GS_CUDA(cudaMemcpyAsync(tile_ranges, ctx->ranges, (size_t)ctx->cam.tiles_x * ctx->cam.tiles_y * 8, cudaMemcpyDeviceToDevice, s));
  return GS_OK;
}

int gs_get_features(gs_ctx* ctx, void* stream, double* mean2d, float* conic, float* color, float* depth,
                    uint32_t* depth_key, int32_t* rect) {
  if (!ctx) return GS_E_INVALID;
  if (ctx->stage < 1) return fail(ctx, GS_E_ORDER, "gs_get_features before gs_preprocess");
  GS_CUDA(cudaSetDevice(ctx->device));
  if (ctx->N == 0) return GS_OK;
  features_export_kernel<<<(unsigned)div_up(ctx->N, 256), 256, 0, (cudaStream_t)stream>>>(
      ctx->N, ctx->feat, ctx->vis_rec, ctx->tiles_touched, ctx->slot_of, mean2d, conic, color, depth, depth_key,
      rect);
  GS_LAUNCH_CHECK("features_export_kernel");
  return GS_OK;
}

int gs_profile_enable(gs_ctx* ctx, int on) {
  if (!ctx) return GS_E_INVALID;
  GS_CUDA(cudaSetDevice(ctx->device));
  if (on && !ctx->ev_made) {
    for (int k = 0; k < 13; ++k) GS_CUDA(cudaEventCreate(&ctx->ev[k]));
    ctx->ev_made = true;
  }
  ctx->prof_on = on != 0;
  return GS_OK;
}

int gs_profile_read(gs_ctx* ctx, float* ms) {
  if (!ctx || !ms) return GS_E_INVALID;
  if (!ctx->prof_on) return fail(ctx, GS_E_ORDER, "gs_profile_read: profiling is not enabled");
  GS_CUDA(cudaSetDevice(ctx->device));
  GS_CUDA(cudaEventSynchronize(ctx->ev[12]));
  static const int from[GS_NUM_STAGES] = {0, 2, 3, 4, 6, 8, 9, 11};
  static const int to[GS_NUM_STAGES] = {1, 3, 4, 5, 7, 9, 10, 12};
  for (int k = 0; k < GS_NUM_STAGES; ++k) GS_CUDA(cudaEventElapsedTime(&ms[k], ctx->ev[from[k]], ctx->ev[to[k]]));
  return GS_OK;
}

int gs_get_launch_count(gs_ctx* ctx, uint64_t* n) {
  if (!ctx || !n) return GS_E_INVALID;
  *n = ctx->launches;
  return GS_OK;
}

int gs_get_workload(gs_ctx* ctx, void* stream, uint64_t* out) {
  if (!ctx || !out) return GS_E_INVALID;
  if (ctx->stage < 3) return fail(ctx, GS_E_ORDER, "gs_get_workload before gs_rasterize_fwd");
  GS_CUDA(cudaSetDevice(ctx->device));
  return launch_workload_stats(ctx, (cudaStream_t)stream, out);
}

int gs_aux_l1_grad(void* stream, int64_t n, const float* pred, const float* target, float weight, float* grad) {
  if (n < 0 || (n > 0 && (!pred || !target || !grad))) return GS_E_INVALID;
  if (n == 0) return GS_OK;
  l1_grad_kernel<<<(unsigned)div_up(n, 256), 256, 0, (cudaStream_t)stream>>>(n, pred, target, weight, grad);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

int gs_aux_pose_step(void* stream, float* T_cw_dev, const float* g_twist, float step) {
  if (!T_cw_dev || !g_twist) return GS_E_INVALID;
  pose_step_kernel<<<1, 32, 0, (cudaStream_t)stream>>>(T_cw_dev, g_twist, step);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

int gs_refine_views(gs_ctx* ctx, void* stream, int64_t N, int sh_degree, const gs_gaussians* params,
                    const gs_refine_batch* batch, const float* bg, const gs_gaussians* grads, float* g_twist, float* g_ab,
                    double* loss, uint32_t* visible) {
  if (!ctx) return GS_E_INVALID;
  if (!params || !batch || !grads || !g_twist || !g_ab || !loss || batch->n_views < 1 || !batch->cams || !batch->target_rgb ||
      !batch->target_depth || !batch->ab)
    return fail(ctx, GS_E_INVALID, "gs_refine_views: null argument or no view");
  const int32_t W = batch->cams[0].width, H = batch->cams[0].height;
  for (int v = 0; v < batch->n_views; ++v)
    if (batch->cams[v].width != W || batch->cams[v].height != H) return fail(ctx, GS_E_INVALID, "gs_refine_views: views differ in size");
  if (W <= 0 || H <= 0) return fail(ctx, GS_E_INVALID, "gs_refine_views: empty image");
  cudaStream_t s = (cudaStream_t)stream;
  GS_CUDA(cudaSetDevice(ctx->device));
  // an overflow left by an earlier call on ANY of the contexts involved is reported before anything is enqueued
  { const int rc = handle_overflow_all(ctx); if (rc != GS_OK) return rc; }
  const int64_t P = (int64_t)W * H;
  // GS_OPT_VIEW_STREAMS > 1: the views run round-robin on this context (caller's stream) and on S - 1 sub-contexts with
  // their own streams; every view ACCUMULATES (one L2 reduction per element) into gradient arrays zeroed up front, so the
  // order in which the views finish does not matter.  S == 1: view 0 writes, the others accumulate, all on `stream`.
  const int S = std::min(ctx->opt_view_streams, batch->n_views);
  for (int k = 0; k + 1 < S; ++k) {
    if (!ctx->sub[k]) {
      int rc = gs_create(&ctx->sub[k], ctx->device);
      if (rc != GS_OK) return fail(ctx, rc, "gs_refine_views: could not create a sub-context");
      ctx->sub[k]->opt_exact_cull = ctx->opt_exact_cull;
      GS_CUDA(cudaStreamCreateWithFlags(&ctx->sub_stream[k], cudaStreamNonBlocking));
      GS_CUDA(cudaEventCreateWithFlags(&ctx->ev_view_join[k], cudaEventDisableTiming));
    }
  }
  if (S > 1 && !ctx->ev_view_fork) GS_CUDA(cudaEventCreateWithFlags(&ctx->ev_view_fork, cudaEventDisableTiming));
  for (int k = 0; k < S; ++k) {
    gs_ctx* c = k == 0 ? ctx : ctx->sub[k - 1];
    if (18 * P > c->rv_floats) {   // rendered rgb (3), depth, alpha, d_rgb (3), d_depth, SSIM scratch (9)
      GS_CUDA(cudaDeviceSynchronize());
      int rc = grow(c, c->rv, 18 * P);
      if (rc != GS_OK) { c->rv_floats = 0; return fail(ctx, rc, "gs_refine_views: out of memory"); }
      c->rv_floats = 18 * P;
    }
  }
  if (visible && N > 0) GS_CUDA(cudaMemsetAsync(visible, 0, (size_t)N * sizeof(uint32_t), s));
  if (S > 1) {
    const int64_t K3 = 3 * (int64_t)(sh_degree + 1) * (sh_degree + 1);
    if (N > 0) {
      GS_CUDA(cudaMemsetAsync(grads->means, 0, (size_t)N * 3 * sizeof(float), s));
      GS_CUDA(cudaMemsetAsync(grads->scales, 0, (size_t)N * 3 * sizeof(float), s));
      GS_CUDA(cudaMemsetAsync(grads->quats, 0, (size_t)N * 4 * sizeof(float), s));
      GS_CUDA(cudaMemsetAsync(grads->opacities, 0, (size_t)N * sizeof(float), s));
      GS_CUDA(cudaMemsetAsync(grads->sh, 0, (size_t)N * K3 * sizeof(float), s));
    }
    GS_CUDA(cudaEventRecord(ctx->ev_view_fork, s));
    for (int k = 0; k + 1 < S; ++k) GS_CUDA(cudaStreamWaitEvent(ctx->sub_stream[k], ctx->ev_view_fork, 0));
  }
  int rc_all = GS_OK;
  for (int v = 0; v < batch->n_views && rc_all == GS_OK; ++v) {
    const int k = v % S;
    gs_ctx* c = k == 0 ? ctx : ctx->sub[k - 1];
    cudaStream_t vs = k == 0 ? s : ctx->sub_stream[k - 1];
    void* vstream = (void*)vs;
    float *rgb = c->rv, *depth = rgb + 3 * P, *alpha = depth + P, *d_rgb = alpha + P, *d_depth = d_rgb + 3 * P, *work = d_depth + P;
    int rc;
    auto view = [&]() -> int {
      const float* T_dev = batch->T_cw_dev ? batch->T_cw_dev + 12 * v : nullptr;
      if ((rc = gs_preprocess(c, vstream, N, sh_degree, params->means, params->scales, params->quats, params->opacities,
                              params->sh, &batch->cams[v], T_dev)) != GS_OK) return rc;
      if ((rc = gs_bin_tiles(c, vstream)) != GS_OK) return rc;
      if ((rc = gs_rasterize_fwd(c, vstream, bg, rgb, depth, alpha)) != GS_OK) return rc;
      double* lv = loss + 10 * v;
      if ((rc = gs_loss_refine(vstream, W, H, rgb, depth, batch->target_rgb + 3 * P * v, batch->target_depth + P * v,
                               batch->ab + 2 * v, batch->alpha_p, batch->lambda, batch->beta, d_rgb, d_depth, g_ab + 2 * v, work,
                               lv)) != GS_OK) return fail(c, rc, "gs_refine_views: gs_loss_refine failed");
      if (batch->normal_prior) {
        const gs_camera& cm = batch->cams[v];
        if ((rc = gs_loss_normal(vstream, W, H, cm.fx, cm.fy, cm.cx, cm.cy, depth, batch->normal_prior + 3 * P * v, batch->lambda_n,
                                 nullptr, d_depth, lv + 8)) != GS_OK) return fail(c, rc, "gs_refine_views: gs_loss_normal failed");
      } else {
        if (cudaMemsetAsync(lv + 8, 0, 2 * sizeof(double), vs) != cudaSuccess) return GS_E_CUDA;
      }
      if ((rc = gs_rasterize_bwd(c, vstream, d_rgb, d_depth, nullptr, (S > 1 || v > 0) ? GS_ACCUMULATE : 0u, grads->means,
                                 grads->scales, grads->quats, grads->opacities, grads->sh)) != GS_OK) return rc;
      if ((rc = gs_pose_grad(c, vstream, 0u, g_twist + 6 * v)) != GS_OK) return rc;
      if (visible && N > 0) {
        visible_or_kernel<<<(unsigned)div_up(N, 256), 256, 0, vs>>>(N, c->tiles_touched, visible);
        if (cudaGetLastError() != cudaSuccess) return GS_E_CUDA;
        c->launches++;
      }
      return GS_OK;
    };
    rc_all = view();
    if (rc_all != GS_OK && c != ctx) snprintf(ctx->err, sizeof(ctx->err), "%s", c->err);
  }
  // join: the caller's stream waits for the sub-streams (also after an error, so that nothing is left running unordered)
  for (int k = 0; k + 1 < S; ++k) {
    GS_CUDA(cudaEventRecord(ctx->ev_view_join[k], ctx->sub_stream[k]));
    GS_CUDA(cudaStreamWaitEvent(s, ctx->ev_view_join[k], 0));
  }
  return rc_all;
}

static int fwd_bwd_host(gs_ctx* ctx, void* stream, int64_t N, int sh_degree, const float* means, const float* scales,
                        const float* quats, const float* opacities, const float* sh, const gs_camera* cam, const float* bg,
                        const float* d_rgb, const float* d_depth, float* rgb, float* depth, float* alpha, float* g_means,
                        float* g_scales, float* g_quats, float* g_opacities, float* g_sh, float* g_twist, bool sync) {
  if (!ctx || !cam || sh_degree < 0 || sh_degree > 3 || N < 0) return GS_E_INVALID;
  if (!d_rgb) return fail(ctx, GS_E_INVALID, "gs_fwd_bwd_host: d_rgb is null");
  cudaStream_t s = (cudaStream_t)stream;
  GS_CUDA(cudaSetDevice(ctx->device));
  const int64_t K3 = 3 * (sh_degree + 1) * (sh_degree + 1);
  const int64_t P = (int64_t)cam->width * cam->height;
  auto al = [](int64_t v) { return (v + 63) / 64 * 64; };  // keep every sub-array 256-byte aligned
  const int64_t need = 2 * (2 * al(N * 3) + al(N * 4) + al(N) + al(N * K3)) + 2 * al(3 * P) + 3 * al(P) + al(8);
  if (need > ctx->hb_floats) {
    GS_CUDA(cudaDeviceSynchronize());
    int rc = grow(ctx, ctx->hb, need);
    if (rc != GS_OK) { ctx->hb_floats = 0; return rc; }
    ctx->hb_floats = need;
  }
  float* p = ctx->hb;
  auto take = [&](int64_t n) { float* r = p; p += al(n); return r; };
  float *d_means = take(N * 3), *d_scales = take(N * 3), *d_quats = take(N * 4), *d_opac = take(N), *d_sh = take(N * K3);
  float *dg_means = take(N * 3), *dg_scales = take(N * 3), *dg_quats = take(N * 4), *dg_opac = take(N), *dg_sh = take(N * K3);
  float *d_drgb = take(3 * P), *d_ddepth = take(P), *d_rgb_o = take(3 * P), *d_depth_o = take(P), *d_alpha_o = take(P);
  float* d_twist = take(8);
  const size_t f = sizeof(float);
  if (N > 0) {
    GS_CUDA(cudaMemcpyAsync(d_means, means, N * 3 * f, cudaMemcpyHostToDevice, s));
    GS_CUDA(cudaMemcpyAsync(d_scales, scales, N * 3 * f, cudaMemcpyHostToDevice, s));
    GS_CUDA(cudaMemcpyAsync(d_quats, quats, N * 4 * f, cudaMemcpyHostToDevice, s));
    GS_CUDA(cudaMemcpyAsync(d_opac, opacities, N * f, cudaMemcpyHostToDevice, s));
    GS_CUDA(cudaMemcpyAsync(d_sh, sh, N * K3 * f, cudaMemcpyHostToDevice, s));
  }
  GS_CUDA(cudaMemcpyAsync(d_drgb, d_rgb, 3 * P * f, cudaMemcpyHostToDevice, s));
  if (d_depth) GS_CUDA(cudaMemcpyAsync(d_ddepth, d_depth, P * f, cudaMemcpyHostToDevice, s));
  int rc;
  if ((rc = gs_preprocess(ctx, stream, N, sh_degree, d_means, d_scales, d_quats, d_opac, d_sh, cam, nullptr)) != GS_OK) return rc;
  if ((rc = gs_bin_tiles(ctx, stream)) != GS_OK) return rc;
  if ((rc = gs_rasterize_fwd(ctx, stream, bg, d_rgb_o, d_depth_o, d_alpha_o)) != GS_OK) return rc;
  if ((rc = gs_rasterize_bwd(ctx, stream, d_drgb, d_depth ? d_ddepth : nullptr, nullptr, 0, dg_means, dg_scales, dg_quats,
                             dg_opac, dg_sh)) != GS_OK) return rc;
  if ((rc = gs_pose_grad(ctx, stream, 0, d_twist)) != GS_OK) return rc;
  if (rgb) GS_CUDA(cudaMemcpyAsync(rgb, d_rgb_o, 3 * P * f, cudaMemcpyDeviceToHost, s));
  if (depth) GS_CUDA(cudaMemcpyAsync(depth, d_depth_o, P * f, cudaMemcpyDeviceToHost, s));
  if (alpha) GS_CUDA(cudaMemcpyAsync(alpha, d_alpha_o, P * f, cudaMemcpyDeviceToHost, s));
  if (N > 0) {
    if (g_means) GS_CUDA(cudaMemcpyAsync(g_means, dg_means, N * 3 * f, cudaMemcpyDeviceToHost, s));
    if (g_scales) GS_CUDA(cudaMemcpyAsync(g_scales, dg_scales, N * 3 * f, cudaMemcpyDeviceToHost, s));
    if (g_quats) GS_CUDA(cudaMemcpyAsync(g_quats, dg_quats, N * 4 * f, cudaMemcpyDeviceToHost, s));
    if (g_opacities) GS_CUDA(cudaMemcpyAsync(g_opacities, dg_opac, N * f, cudaMemcpyDeviceToHost, s));
    if (g_sh) GS_CUDA(cudaMemcpyAsync(g_sh, dg_sh, N * K3 * f, cudaMemcpyDeviceToHost, s));
  }
  if (g_twist) GS_CUDA(cudaMemcpyAsync(g_twist, d_twist, 6 * f, cudaMemcpyDeviceToHost, s));
  if (!sync) return GS_OK;
  GS_CUDA(cudaStreamSynchronize(s));
  return gs_poll(ctx);
}

int gs_fwd_bwd_host(gs_ctx* ctx, void* stream, int64_t N, int sh_degree, const float* means, const float* scales,
                    const float* quats, const float* opacities, const float* sh, const gs_camera* cam, const float* bg,
                    const float* d_rgb, const float* d_depth, float* rgb, float* depth, float* alpha, float* g_means,
                    float* g_scales, float* g_quats, float* g_opacities, float* g_sh, float* g_twist) {
  return fwd_bwd_host(ctx, stream, N, sh_degree, means, scales, quats, opacities, sh, cam, bg, d_rgb, d_depth, rgb, depth,
                      alpha, g_means, g_scales, g_quats, g_opacities, g_sh, g_twist, true);
}

int gs_fwd_bwd_host_async(gs_ctx* ctx, void* stream, int64_t N, int sh_degree, const float* means, const float* scales,
                          const float* quats, const float* opacities, const float* sh, const gs_camera* cam,
                          const float* bg, const float* d_rgb, const float* d_depth, float* rgb, float* depth, float* alpha,
                          float* g_means, float* g_scales, float* g_quats, float* g_opacities, float* g_sh, float* g_twist) {
  return fwd_bwd_host(ctx, stream, N, sh_degree, means, scales, quats, opacities, sh, cam, bg, d_rgb, d_depth, rgb, depth,
                      alpha, g_means, g_scales, g_quats, g_opacities, g_sh, g_twist, false);
}

}  // extern "C"

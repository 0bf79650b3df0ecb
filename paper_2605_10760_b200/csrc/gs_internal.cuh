// gs_internal.cuh -- context, device-side records and small helpers shared by the CUDA translation units of libgs.so.
// Product code: nothing here (or in any file of csrc/) includes, links or calls oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/gs.h"

namespace gs {

// ---------------------------------------------------------------------------------------------------------------
// Device-side camera (kernel argument, by value).  `T_dev` non-null overrides `T` (pose updated on the device).
// ---------------------------------------------------------------------------------------------------------------
struct DevCam {
  int32_t W, H, tiles_x, tiles_y;
  float fx, fy, cx, cy, near_z;
  float T[12];
  const float* T_dev;
};

__device__ __forceinline__ void load_pose(const DevCam& cam, float* T) {
  if (cam.T_dev) {
#pragma unroll
    for (int k = 0; k < 12; ++k) T[k] = __ldg(cam.T_dev + k);
  } else {
#pragma unroll
    for (int k = 0; k < 12; ++k) T[k] = cam.T[k];
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Per-Gaussian feature record written by gs_preprocess, indexed by visible slot: 3 x float4 = 48 B.
//   f0 = { mfx, mfy, bits(miy << 16 | mix & 0xffff), opacity }  2-D mean = integer pixel (mix,miy) + fraction in [-0.5,0.5]
//   f1 = { l11, l21, l22, lo }  L = sqrt(0.5 log2 e) chol(conic) (lower triangular, fp64 in gs_preprocess), lo = log2(opacity):
//                               p2(d) = lo - (l11 dx + l21 dy)^2 - (l22 dy)^2,  alpha = min(0.99, 2^p2),
//                               alpha >= 1/255  <=>  p2 >= -log2(255)            (gs_raster.cuh)
//   f2 = { r, g, b, z_c }
// f1, f2 (32 contiguous bytes) are what the compositing kernels gather; f0 is read by the binning kernels only.
// Per tile INSTANCE (sorted list position) gs_bin_tiles also writes uv = (u0, v0) = -L^T (mean - tile origin), formed in
// fp64: with it the per-pixel arithmetic of the compositing kernels is u = l11 X + l21 Y + u0, v = l22 Y + v0 on
// tile-local pixel coordinates (X, Y) in 0..15 -- every operand O(10), whatever the footprint.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kFeatVec = 3;

// 2-D gradient record accumulated by the pixel backward (global atomics), 12 floats = 48 B per Gaussian: moments of
// gp = alpha * dL/dalpha (unclamped contributions) in the WHITENED offsets (u, v) = L^T (pixel - mean) of gs_raster.cuh
//   [0] sum gp u                [1] sum gp v                [2] sum gp u^2    [3] sum gp u v     [4] sum gp v^2
//   [5] sum gp                  [6..8] sum w gC             [9] sum w gD      [10],[11] unused          (w = alpha T)
// from which dL/dmean = L M1 / k and dL/dSigma' = L M2 L^T / (2 k^2), k = 0.5 log2(e)  (gs_gauss_bwd.cu).
constexpr int kG2D = 12;

// Programmatic dependent launch (sm_90+): every kernel of the iteration is launched with
// cudaLaunchAttributeProgrammaticStreamSerialization and starts with pdl_enter(): griddepcontrol.wait returns once the
// kernel in front of it in the stream has completed and its writes are visible (every CTA of every kernel calls it
// unconditionally, so completion is transitive along the chain), launch_dependents then lets the CTAs of the NEXT kernel
// become resident while this one drains: launch latency and the ramp of each kernel hide under the tail of the one
// before.  Without the launch attribute both instructions are no-ops.
__device__ __forceinline__ void pdl_enter() {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

// Header allocation: two Counts records (64 B apart; iteration seq uses record seq & 1, so the count of visible Gaussians
// of one iteration stays readable until the next gs_preprocess while the other record is already cleared for it) + 16 pose
// accumulators, in front of the per-tile counters (gs_api.cu).  Steady state needs no memset: tile_scan_kernel clears the
// tile counters it has read and the other Counts record, preprocess_kernel clears the pose accumulators.
constexpr int kHdrBytes = 256;
#ifndef GS_CTR_STRIDE
#define GS_CTR_STRIDE 32
#endif
constexpr int kCtrStride = GS_CTR_STRIDE;  // per-tile counters are one per 128-byte line (gs_binning.cu)

// Device counters (one per context) + pinned-host mirror ("mailbox") the host may poll without synchronising.
struct alignas(16) Counts {
  uint32_t n_visible;
  uint32_t n_instances;  // total tile instances of the last scan (even if it overflowed)
  uint32_t overflow;     // 1 if n_instances > capacity: nothing was emitted and downstream kernels see 0 instances
  uint32_t seq;          // iteration number of the writer
  uint32_t n_large;      // number of tiles whose list is longer than one 4-warp CTA sorts in registers (> 2047)
  uint32_t n_mid;        // number of tiles whose list is longer than one warp sorts in registers (> 255; includes n_large)
};


}  // namespace gs

// ---------------------------------------------------------------------------------------------------------------
// Host-side context
// ---------------------------------------------------------------------------------------------------------------
struct gs_ctx {
  int device = 0;
  char err[512] = {0};

  // last gs_preprocess
  int64_t N = 0;
  int sh_degree = 0;
  gs::DevCam cam{};
  const float *means = nullptr, *scales = nullptr, *quats = nullptr, *opacities = nullptr, *sh = nullptr;
  int stage = 0;  // 0 nothing, 1 preprocessed, 2 binned, 3 rasterised fwd, 4 backward done
  uint32_t seq = 0;
  float bg[3] = {0, 0, 0};

  // per-Gaussian scratch (capacity cap_N)
  int64_t cap_N = 0;
  float4* feat = nullptr;           // [N,3], indexed by VISIBLE SLOT
  uint32_t* tiles_touched = nullptr;  // [N]
  uint32_t* vis_ids = nullptr;        // [N] indices of the visible Gaussians, compacted (arbitrary order)
  uint4* vis_rec = nullptr;           // [N] same order: {tx0 | ty0 << 16, tx1 | ty1 << 16, depth key, index}
  float4* vis_par = nullptr;          // [N,3] same order: {mu, opacity} {scale, -} {quat}: what gauss_bwd needs again
  uint32_t* slot_of = nullptr;        // [N] visible slot of Gaussian i (valid where tiles_touched[i] > 0)
  float* g2d = nullptr;             // [N,12], indexed by visible slot; kept all-zero between iterations (the consumer clears what it reads)
  bool g2d_dirty = false;

  // per-instance scratch (capacity cap_I)
  int64_t cap_I = 0;
  bool calibrated = false;
  int64_t cal_N = -1;
  int32_t cal_W = -1, cal_H = -1;
  uint64_t* keys[2] = {nullptr, nullptr};  // [0]: (depth bits << 32 | id) bucketed by tile, sorted in place
  // [cap_I] one 16-byte record per sorted instance, what the compositing kernels stage with a single cp.async:
  // {u0, v0, bits(visible slot << 8 | region mask), -}: the whitened tile-local offset of the instance and its list word
  float4* inst_rec = nullptr;
  int sorted_buf = 0;
  bool sort_attr_set = false;

  // per-tile / per-pixel scratch
  int64_t cap_tiles = 0, cap_pix = 0;
  uint2* ranges = nullptr;          // [tiles]
  uint32_t* tile_count = nullptr;   // [tiles] instances per tile (atomics in gs_preprocess)
  uint32_t* tile_cursor = nullptr;  // [tiles] write cursors of the duplication
  uint32_t* scan_ws = nullptr;      // tile scan: per-CTA totals [128][17] as 64-bit words {epoch, value}
  uint32_t scan_epoch = 0;
  bool scan_pdl = true;             // the cooperative tile scan also takes the programmatic-serialization attribute
  float* final_T = nullptr;         // [H*W]
  uint32_t* n_contrib = nullptr;    // [H*W]

  // pose-gradient accumulators: 15 doubles: sum g_pc (3), sum g_v (3), g_W (9)
  double* pose_acc = nullptr;
  bool pose_acc_valid = false;
  bool pose_acc_clean = false;  // zeroed by gs_preprocess and not yet accumulated into
  unsigned long long* stats_ws = nullptr;  // gs_get_workload: its own 8 counters (never the pose accumulators)
  char* hdr = nullptr;          // one allocation: counts x 2, pose_acc, tile_count
  bool hdr_clean = false;       // the tile counters and the Counts record of the NEXT iteration are zero (else: one memset)
  int64_t ctr_dirty = 0;        // number of leading tile counters that may be non-zero (image sizes may change between calls)

  gs::Counts* counts = nullptr;       // device
  gs::Counts* mailbox = nullptr;      // pinned host, mapped
  gs::Counts* mailbox_dev = nullptr;  // device alias of the mailbox

  uint32_t* tile_order = nullptr;      // [tiles] tile ids by descending list length (longest lists are scheduled first)
  bool opt_exact_cull = false;         // GS_OPT_EXACT_TILE_CULL (gs_set_option)
  // GS_OPT_VIEW_STREAMS (gs_set_option): gs_refine_views issues its views round-robin on this context and on
  // opt_view_streams - 1 context-owned sub-contexts with their own streams (created on first use)
  int opt_view_streams = 1;
  gs_ctx* sub[7] = {};
  cudaStream_t sub_stream[7] = {};
  cudaEvent_t ev_view_fork = nullptr, ev_view_join[7] = {};

  // side stream: the block-wide sort of the few long tile lists runs beside the warp-level sort of the rest
  cudaStream_t side_stream = nullptr;
  cudaEvent_t ev_fork2 = nullptr, ev_join2 = nullptr;

  // stage timing (gs_profile_*): events recorded around the kernel groups when enabled
  bool prof_on = false;
  cudaEvent_t ev[13] = {};
  bool ev_made = false;
  uint64_t launches = 0;  // kernels launched by this context (gs_get_launch_count)

  // gs_refine_views: rendered images, upstream gradients and SSIM scratch of one view (18 H W floats), grown on demand
  float* rv = nullptr;
  int64_t rv_floats = 0;

  // host-buffer path (gs_fwd_bwd_host): device staging, grown on demand
  float* hb = nullptr;
  int64_t hb_floats = 0;
};

namespace gs {

inline int fail(gs_ctx* ctx, int code, const char* msg) {
  if (ctx) snprintf(ctx->err, sizeof(ctx->err), "%s", msg);
  return code;
}

inline int fail_cuda(gs_ctx* ctx, cudaError_t e, const char* where) {
  if (ctx) snprintf(ctx->err, sizeof(ctx->err), "%s: %s", where, cudaGetErrorString(e));
  return GS_E_CUDA;
}

#define GS_CUDA(call)                                                  \
  do {                                                                 \
    cudaError_t e__ = (call);                                          \
    if (e__ != cudaSuccess) return gs::fail_cuda(ctx, e__, #call);     \
  } while (0)

#define GS_LAUNCH_CHECK(name)                                          \
  do {                                                                 \
    cudaError_t e__ = cudaGetLastError();                              \
    if (e__ != cudaSuccess) return gs::fail_cuda(ctx, e__, name);      \
    ctx->launches++;                                                   \
  } while (0)

// Launch with the programmatic-stream-serialization attribute (see pdl_enter above).
#define GS_LAUNCH_PDL(kernel, grid__, block__, smem__, stream__, ...)                                         \
  do {                                                                                                 \
    cudaLaunchConfig_t cfg__ = {};                                                                     \
    cfg__.gridDim = dim3(grid__); cfg__.blockDim = dim3(block__);                                          \
    cfg__.dynamicSmemBytes = (smem__); cfg__.stream = (stream__);                                          \
    cudaLaunchAttribute at__[1];                                                                       \
    at__[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;                                   \
    at__[0].val.programmaticStreamSerializationAllowed = 1;                                            \
    cfg__.attrs = at__; cfg__.numAttrs = 1;                                                            \
    GS_CUDA(cudaLaunchKernelEx(&cfg__, kernel, __VA_ARGS__));                                          \
  } while (0)

// stage-timing event k on stream s (no-op unless gs_profile_enable(ctx, 1))
#define GS_PROF(k, s)                                                  \
  do {                                                                 \
    if (ctx->prof_on) cudaEventRecord(ctx->ev[k], s);                  \
  } while (0)

// Replaces the buffer by one of `count` elements (contents are not kept).  The new buffer is allocated FIRST and
// swapped in on success: when cudaMalloc fails the old buffer -- and the capacity the caller recorded for it -- stay valid.
template <typename T>
inline int grow(gs_ctx* ctx, T*& p, int64_t count) {
  T* fresh = nullptr;
  if (count > 0) {
    cudaError_t e = cudaMalloc((void**)&fresh, (size_t)count * sizeof(T));
    if (e != cudaSuccess) {
      cudaGetLastError();
      return fail(ctx, GS_E_NOMEM, "cudaMalloc failed while growing scratch");
    }
  }
  if (p) cudaFree(p);
  p = fresh;
  return GS_OK;
}

inline int64_t div_up(int64_t a, int64_t b) { return (a + b - 1) / b; }

// Non-blocking read of the pinned-host mailbox the device writes.
inline Counts read_mailbox(const gs_ctx* ctx) {
  // the device writes the first four words with one 16-byte store; re-read until the sequence word is stable
  const volatile Counts* m = ctx->mailbox;
  Counts c;
  for (int attempt = 0; attempt < 4; ++attempt) {
    c.seq = m->seq;
    c.n_visible = m->n_visible; c.n_instances = m->n_instances; c.overflow = m->overflow;
    if (m->seq == c.seq) break;
  }
  c.n_large = m->n_large;  // a hint only (written by a second store)
  c.n_mid = 0;
  return c;
}

// entry points implemented across translation units
int launch_preprocess(gs_ctx* ctx, cudaStream_t s);
int launch_binning(gs_ctx* ctx, cudaStream_t s);
int launch_raster_fwd(gs_ctx* ctx, cudaStream_t s, float* rgb, float* depth, float* alpha);
int launch_raster_bwd(gs_ctx* ctx, cudaStream_t s, const float* d_rgb, const float* d_depth, const float* d_alpha);
int launch_gauss_bwd(gs_ctx* ctx, cudaStream_t s, uint32_t flags, float* g_means, float* g_scales, float* g_quats,
                     float* g_opac, float* g_sh);
int launch_pose_final(gs_ctx* ctx, cudaStream_t s, uint32_t flags, float* g_twist);
int ensure_instance_capacity(gs_ctx* ctx, int64_t need);
int handle_overflow(gs_ctx* ctx);
int export_sorted_keys(gs_ctx* ctx, cudaStream_t s, uint64_t* out);
int export_sorted_ids(gs_ctx* ctx, cudaStream_t s, int64_t I, uint32_t* out);
int launch_workload_stats(gs_ctx* ctx, cudaStream_t s, uint64_t* out_host);

}  // namespace gs

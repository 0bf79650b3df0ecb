// gs_raster.cu -- steps a6 (front-to-back compositing) and a8 (back-to-front per-pixel backward with warp-level
// reduction before global atomics).  One CTA per 16x16 tile, one thread per pixel, Gaussians staged through shared
// memory in batches of 256.  ALU/MUFU-bound.
#include "gs_internal.cuh"
#include "gs_raster.cuh"

namespace gs {

__global__ void __launch_bounds__(kBatch)
raster_fwd_kernel(int W, int H, int tiles_x, const uint2* __restrict__ ranges, const uint32_t* __restrict__ ids,
                  const float4* __restrict__ feat, float bg0, float bg1, float bg2, float* __restrict__ rgb,
                  float* __restrict__ depth, float* __restrict__ alpha_out, float* __restrict__ final_T,
                  uint32_t* __restrict__ n_contrib) {
  __shared__ Staged sm[kBatch];
  const int tile = blockIdx.x;
  const int ox = (tile % tiles_x) * GS_TILE, oy = (tile / tiles_x) * GS_TILE;
  int lx, ly;
  thread_pixel(threadIdx.x, lx, ly);
  const int px = ox + lx, py = oy + ly;
  const bool inside = px < W && py < H;
  const float fx = (float)lx, fy = (float)ly;
  const uint2 range = ranges[tile];
  const int n = (int)(range.y - range.x);
  float T = 1.f, C0 = 0.f, C1 = 0.f, C2 = 0.f, D = 0.f;
  uint32_t last = 0;
  bool done = !inside;
  for (int b0 = 0; b0 < n; b0 += kBatch) {
    if (__syncthreads_and(done)) break;
    const int idx = b0 + threadIdx.x;
    if (idx < n) stage_gaussian(feat, __ldg(ids + range.x + idx), ox, oy, sm[threadIdx.x]);
    __syncthreads();
    if (__all_sync(0xffffffffu, done)) continue;
    const int cnt = min(kBatch, n - b0);
    for (int j = 0; j < cnt && !done; ++j) {
      const float4 g0 = sm[j].g0, g1 = sm[j].g1;
      const float dx = fx - g0.x, dy = fy - g0.y;
      const float og = eval_og(dx, dy, g0.z, g0.w, g1.x, g1.y);
      const float a = fminf(GS_ALPHA_MAX, og);
      if (a < GS_ALPHA_MIN) continue;
      if (T < GS_T_MIN) { done = true; break; }
      const float4 g2 = sm[j].g2;
      const float w = a * T;
      C0 = fmaf(g1.z, w, C0);
      C1 = fmaf(g1.w, w, C1);
      C2 = fmaf(g2.x, w, C2);
      D = fmaf(g2.y, w, D);
      T = T * (1.f - a);
      last = (uint32_t)(b0 + j + 1);
    }
  }
  if (inside) {
    const size_t p = (size_t)py * W + px, HW = (size_t)W * H;
    if (rgb) {
      rgb[p] = fmaf(T, bg0, C0);
      rgb[HW + p] = fmaf(T, bg1, C1);
      rgb[2 * HW + p] = fmaf(T, bg2, C2);
    }
    if (depth) depth[p] = D;
    if (alpha_out) alpha_out[p] = 1.f - T;
    final_T[p] = T;
    n_contrib[p] = last;
  }
}

__global__ void __launch_bounds__(kBatch)
raster_bwd_kernel(int W, int H, int tiles_x, const uint2* __restrict__ ranges, const uint32_t* __restrict__ ids,
                  const float4* __restrict__ feat, float bg0, float bg1, float bg2, const float* __restrict__ final_T,
                  const uint32_t* __restrict__ n_contrib, const float* __restrict__ d_rgb,
                  const float* __restrict__ d_depth, const float* __restrict__ d_alpha, float* __restrict__ g2d) {
  __shared__ Staged sm[kBatch];
  __shared__ uint32_t s_max[kBatch / 32];
  const int tile = blockIdx.x;
  const int ox = (tile % tiles_x) * GS_TILE, oy = (tile / tiles_x) * GS_TILE;
  int lx, ly;
  thread_pixel(threadIdx.x, lx, ly);
  const int px = ox + lx, py = oy + ly;
  const bool inside = px < W && py < H;
  const float fx = (float)lx, fy = (float)ly;
  const uint2 range = ranges[tile];
  float T = 1.f, gC0 = 0.f, gC1 = 0.f, gC2 = 0.f, gD = 0.f, gA = 0.f;
  uint32_t last = 0;
  if (inside) {
    const size_t p = (size_t)py * W + px, HW = (size_t)W * H;
    T = final_T[p];
    last = n_contrib[p];
    gC0 = d_rgb[p]; gC1 = d_rgb[HW + p]; gC2 = d_rgb[2 * HW + p];
    if (d_depth) gD = d_depth[p];
    if (d_alpha) gA = d_alpha[p];
  }
  float S = T * (gC0 * bg0 + gC1 * bg1 + gC2 * bg2);
  // deepest blended position in the tile
  uint32_t m = __reduce_max_sync(0xffffffffu, last);
  if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = m;
  __syncthreads();
  uint32_t maxc = 0;
#pragma unroll
  for (int w = 0; w < kBatch / 32; ++w) maxc = max(maxc, s_max[w]);
  const int lane = threadIdx.x & 31;
  const int rounds = (int)((maxc + kBatch - 1) / kBatch);
  for (int r = rounds - 1; r >= 0; --r) {
    const int b0 = r * kBatch;
    __syncthreads();
    const int idx = b0 + threadIdx.x;
    if (idx < (int)maxc) stage_gaussian(feat, __ldg(ids + range.x + idx), ox, oy, sm[threadIdx.x]);
    __syncthreads();
    const int cnt = min(kBatch, (int)maxc - b0);
    for (int j = cnt - 1; j >= 0; --j) {
      const uint32_t pos = (uint32_t)(b0 + j);
      const float4 g0 = sm[j].g0, g1 = sm[j].g1;
      const float dx = fx - g0.x, dy = fy - g0.y;
      const float og = eval_og(dx, dy, g0.z, g0.w, g1.x, g1.y);
      const float a = fminf(GS_ALPHA_MAX, og);
      const bool valid = pos < last && a >= GS_ALPHA_MIN;
      if (!__any_sync(0xffffffffu, valid)) continue;
      const float4 g2 = sm[j].g2;
      float v[10];
#pragma unroll
      for (int k = 0; k < 10; ++k) v[k] = 0.f;
      if (valid) {
        const float oma = 1.f - a;
        T = __fdividef(T, oma);  // transmittance in front of this Gaussian
        const float w = a * T;
        const float wi = fmaf(gC0, g1.z, fmaf(gC1, g1.w, fmaf(gC2, g2.x, fmaf(gD, g2.y, gA))));
        const float dalpha = fmaf(T, wi, -__fdividef(S, oma));
        S = fmaf(wi, w, S);
        v[6] = w * gC0; v[7] = w * gC1; v[8] = w * gC2; v[9] = w * gD;
        if (og <= GS_ALPHA_MAX) {
          const float gp = a * dalpha;
          const float A = g0.z, B = g0.w, Cc = g1.x;
          v[0] = gp * fmaf(2.f * A, dx, B * dy);
          v[1] = gp * fmaf(2.f * Cc, dy, B * dx);
          v[2] = gp * dx * dx;
          v[3] = gp * dx * dy;
          v[4] = gp * dy * dy;
          v[5] = gp;
        }
      }
#pragma unroll
      for (int k = 0; k < 10; ++k) {
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], d);
      }
      if (lane == 0) {
        float* g = g2d + (size_t)__float_as_uint(g2.z) * kG2D;
#pragma unroll
        for (int k = 0; k < 10; ++k) atomicAdd(g + k, v[k]);
      }
    }
  }
}

// Workload statistics of the forward (introspection only): re-walks every pixel's list with the forward's decisions.
__global__ void __launch_bounds__(kBatch)
workload_stats_kernel(int W, int H, int tiles_x, const uint2* __restrict__ ranges, const uint32_t* __restrict__ ids,
                      const float4* __restrict__ feat, unsigned long long* __restrict__ out) {
  __shared__ Staged sm[kBatch];
  const int tile = blockIdx.x;
  const int ox = (tile % tiles_x) * GS_TILE, oy = (tile / tiles_x) * GS_TILE;
  int lx, ly;
  thread_pixel(threadIdx.x, lx, ly);
  const bool inside = (ox + lx) < W && (oy + ly) < H;
  const float fx = (float)lx, fy = (float)ly;
  const uint2 range = ranges[tile];
  const int n = (int)(range.y - range.x);
  float T = 1.f;
  unsigned long long evaluated = 0, blended = 0, last = 0;
  bool done = !inside;
  for (int b0 = 0; b0 < n; b0 += kBatch) {
    __syncthreads();
    const int idx = b0 + threadIdx.x;
    if (idx < n) stage_gaussian(feat, __ldg(ids + range.x + idx), ox, oy, sm[threadIdx.x]);
    __syncthreads();
    const int cnt = min(kBatch, n - b0);
    for (int j = 0; j < cnt && !done; ++j) {
      const float4 g0 = sm[j].g0, g1 = sm[j].g1;
      ++evaluated;
      const float a = fminf(GS_ALPHA_MAX, eval_og(fx - g0.x, fy - g0.y, g0.z, g0.w, g1.x, g1.y));
      if (a < GS_ALPHA_MIN) continue;
      if (T < GS_T_MIN) { done = true; break; }
      T = T * (1.f - a);
      ++blended;
      last = (unsigned long long)(b0 + j + 1);
    }
  }
  unsigned long long v[4] = {evaluated, blended, last, inside ? (unsigned long long)n : 0ull};
#pragma unroll
  for (int k = 0; k < 4; ++k) {
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], d);
    if ((threadIdx.x & 31) == 0 && v[k]) atomicAdd(out + k, v[k]);
  }
}

int launch_workload_stats(gs_ctx* ctx, cudaStream_t s, uint64_t* out_host) {
  const int tiles = ctx->cam.tiles_x * ctx->cam.tiles_y;
  unsigned long long* d = reinterpret_cast<unsigned long long*>(ctx->pose_acc);  // 16 doubles of scratch, unused here
  GS_CUDA(cudaMemsetAsync(d, 0, 4 * sizeof(unsigned long long), s));
  if (tiles > 0) {
    workload_stats_kernel<<<tiles, kBatch, 0, s>>>(ctx->cam.W, ctx->cam.H, ctx->cam.tiles_x, ctx->ranges,
                                                   ctx->vals[ctx->sorted_buf], ctx->feat, d);
    GS_LAUNCH_CHECK("workload_stats_kernel");
  }
  GS_CUDA(cudaMemcpyAsync(out_host, d, 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
  GS_CUDA(cudaStreamSynchronize(s));
  ctx->pose_acc_valid = false;
  return GS_OK;
}

int launch_raster_fwd(gs_ctx* ctx, cudaStream_t s, float* rgb, float* depth, float* alpha) {
  const int tiles = ctx->cam.tiles_x * ctx->cam.tiles_y;
  if (tiles == 0) return GS_OK;
  raster_fwd_kernel<<<tiles, kBatch, 0, s>>>(ctx->cam.W, ctx->cam.H, ctx->cam.tiles_x, ctx->ranges,
                                             ctx->vals[ctx->sorted_buf], ctx->feat, ctx->bg[0], ctx->bg[1], ctx->bg[2],
                                             rgb, depth, alpha, ctx->final_T, ctx->n_contrib);
  GS_LAUNCH_CHECK("raster_fwd_kernel");
  return GS_OK;
}

int launch_raster_bwd(gs_ctx* ctx, cudaStream_t s, const float* d_rgb, const float* d_depth, const float* d_alpha) {
  const int tiles = ctx->cam.tiles_x * ctx->cam.tiles_y;
  if (tiles == 0) return GS_OK;
  raster_bwd_kernel<<<tiles, kBatch, 0, s>>>(ctx->cam.W, ctx->cam.H, ctx->cam.tiles_x, ctx->ranges,
                                             ctx->vals[ctx->sorted_buf], ctx->feat, ctx->bg[0], ctx->bg[1], ctx->bg[2],
                                             ctx->final_T, ctx->n_contrib, d_rgb, d_depth, d_alpha, ctx->g2d);
  GS_LAUNCH_CHECK("raster_bwd_kernel");
  return GS_OK;
}

}  // namespace gs

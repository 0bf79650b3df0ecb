// gs_raster.cu -- step a6: per-tile front-to-back compositing (oracle reading C1 step 7).
//
// Design (evidence: profiles/r1_v1_baseline.md, r1_v3_regions.md, r1_v5_masks.md, r2_*.md):
//   * one WARP per 8x4-pixel region of a tile, one pixel per lane, single-warp CTAs: no block barrier, early exit per
//     region, the hardware CTA scheduler balances the very uneven lists (regions are launched longest tile first);
//   * the list entries are (visible slot << 8 | region mask): gs_bin_tiles already decided which regions of the tile a
//     Gaussian can reach.  Lane g looks at entry g of a batch of 32; the relevant ones are compacted (ballot rank) and
//     only their 48-byte records are gathered by cp.async (LDGSTS), one batch ahead of the compute;
//   * every staged record is turned ONCE per (region, Gaussian) into the whitened region-local form of gs_raster.cuh
//     (fp64, lane-parallel, in place); the pixel loop reads it back as three broadcast LDS.128;
//   * the pixel loop is branch-free: every relevant entry is evaluated and blended under a per-lane predicate
//     (alpha_eff = 0 where the pixel is not hit or has terminated), four entries unrolled, one vote per four entries
//     for the early exit; alpha >= 1/255 is tested in the exponent domain against a constant, so rejected pairs cost
//     no MUFU and the opacity never enters the loop: ~20 instructions per relevant (region, Gaussian) entry.
#include "gs_internal.cuh"
#include "gs_raster.cuh"

namespace gs {

// STATS = true: the same walk with the same decisions, counting the workload instead of writing the image
// (gs_get_workload; never on the timed path).
template <bool STATS>
__global__ void __launch_bounds__(32)
raster_fwd_kernel(int W, int H, int tiles_x, const uint32_t* __restrict__ order, const uint2* __restrict__ ranges,
                  const uint32_t* __restrict__ ids, const float4* __restrict__ feat, float bg0, float bg1, float bg2,
                  float* __restrict__ rgb, float* __restrict__ depth, float* __restrict__ alpha_out,
                  float* __restrict__ final_T, uint32_t* __restrict__ n_contrib, unsigned long long* __restrict__ stats) {
  __shared__ __align__(16) float4 s_feat[2][(kWarpBatch + kGroup) * 3];  // records of the relevant entries (cp.async),
  __shared__ uint32_t s_pos[2][kWarpBatch];                               // decoded in place; their list positions + 1
  const int lane = threadIdx.x;
  const int tile = (int)__ldg(order + blockIdx.x / 8), sub = blockIdx.x % 8;
  const int ox = (tile % tiles_x) * GS_TILE + (sub % 2) * 8, oy = (tile / tiles_x) * GS_TILE + (sub / 2) * 4;
  const int lx = lane & 7, ly = lane >> 3;
  const float fx0 = (float)lx, fy0 = (float)ly;
  const bool inside = ox + lx < W && oy + ly < H;
  const uint2 range = ranges[tile];
  const int n = (int)(range.y - range.x);
  const int nb = (n + kWarpBatch - 1) / kWarpBatch;
  // T starts at 0 for a lane outside the image, so such a lane never blends (and writes nothing)
  float T = inside ? 1.f : 0.f, C0 = 0.f, C1 = 0.f, C2 = 0.f, D = 0.f;
  uint32_t last = 0;
  unsigned long long n_eval = 0, n_blend = 0;
  uint32_t rank = 0, last_rank = 0;   // STATS: relevant entries walked so far; rank of the pixel's last blended one

  auto issue = [&](int b, uint32_t v) -> int {
    const bool relevant = (b * kWarpBatch + lane < n) && ((v >> sub) & 1u);
    const unsigned rel = __ballot_sync(kFull, relevant);
    if (relevant) {
      const int r = __popc(rel & ((1u << lane) - 1u));
      const float4* src = feat + 3 * (size_t)(v >> 8);
      float4* dst = &s_feat[b & 1][r * 3];
      cp_async16(dst, src); cp_async16(dst + 1, src + 1); cp_async16(dst + 2, src + 2);
      s_pos[b & 1][r] = (uint32_t)(b * kWarpBatch + lane + 1);
    }
    cp_async_commit();
    return __popc(rel);
  };
  uint32_t v_next = 0;
  int nrel = 0, nrel_next = 0;
  if (nb > 0) {
    nrel_next = issue(0, lane < n ? __ldg(ids + range.x + lane) : 0u);
    if (nb > 1) v_next = (kWarpBatch + lane < n) ? __ldg(ids + range.x + kWarpBatch + lane) : 0u;
  }
  bool stop = !__any_sync(kFull, inside);
  for (int b = 0; b < nb && !stop; ++b) {
    nrel = nrel_next;
    if (b + 1 < nb) {
      nrel_next = issue(b + 1, v_next);
      const int i2 = (b + 2) * kWarpBatch + lane;
      if (b + 2 < nb) v_next = (i2 < n) ? __ldg(ids + range.x + i2) : 0u;
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncwarp();
    if (nrel == 0) continue;
    float4* sf = s_feat[b & 1];
    if (lane < nrel) {  // decode once per (region, Gaussian), in place: whitened region-local record
      const float4 f0 = sf[3 * lane], f1 = sf[3 * lane + 1];
      float u0, v0, mx, my;
      decode_whitened(f0, f1, ox, oy, u0, v0, mx, my);
      sf[3 * lane] = make_float4(u0, v0, f1.x, f1.y);
      sf[3 * lane + 1] = make_float4(f1.z, f0.w, __uint_as_float(s_pos[b & 1][lane]), 0.f);
    }
    if (lane < kGroup) {  // padding records never pass: lo = -inf  =>  p2 = -inf
      sf[3 * (nrel + lane)] = make_float4(0.f, 0.f, 0.f, 0.f);
      sf[3 * (nrel + lane) + 1] = make_float4(0.f, -INFINITY, 0.f, 0.f);
      sf[3 * (nrel + lane) + 2] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    __syncwarp();
    // phase 2: front to back, branch-free
    for (int r0 = 0; r0 < nrel; r0 += kGroup) {
#pragma unroll
      for (int q = 0; q < kGroup; ++q) {
        const float4 a0 = sf[3 * (r0 + q)], a1 = sf[3 * (r0 + q) + 1], f2 = sf[3 * (r0 + q) + 2];
        const float p = eval_power(a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, fx0, fy0);
        const bool alive = T >= GS_T_MIN;
        const bool hit = (p >= GS_POWER_MIN) && alive;   // alpha >= 1/255 and the pixel has not terminated
        const float a = hit ? fminf(GS_ALPHA_MAX, ex2_approx(p)) : 0.f;
        const float w = a * T;
        C0 = fmaf(f2.x, w, C0);
        C1 = fmaf(f2.y, w, C1);
        C2 = fmaf(f2.z, w, C2);
        D = fmaf(f2.w, w, D);
        T = fmaf(-a, T, T);
        last = hit ? __float_as_uint(a1.z) : last;
        if (STATS && r0 + q < nrel) {
          ++rank;
          n_eval += alive ? 1 : 0;
          n_blend += hit ? 1 : 0;
          last_rank = hit ? rank : last_rank;
        }
      }
      if (!__any_sync(kFull, T >= GS_T_MIN)) { stop = true; break; }
    }
    __syncwarp();
  }
  cp_async_wait<0>();
  if (STATS) {
    // gs.h gs_get_workload: E, C, L, list length x pixels, R (forward), Eb, Rb (what the backward must walk: the
    // relevant entries up to the pixel's / the region's last blended one)
    const uint32_t max_rank = __reduce_max_sync(kFull, last_rank);
    unsigned long long v[GS_NUM_WORKLOAD] = {n_eval, n_blend, inside ? last : 0ull, inside ? (unsigned long long)n : 0ull,
                                            lane == 0 ? rank : 0ull, last_rank, lane == 0 ? max_rank : 0ull};
#pragma unroll
    for (int q = 0; q < GS_NUM_WORKLOAD; ++q) {
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) v[q] += __shfl_xor_sync(kFull, v[q], d);
      if (lane == 0 && v[q]) atomicAdd(stats + q, v[q]);
    }
    return;
  }
  if (inside) {
    const size_t HW = (size_t)W * H;
    const size_t p = (size_t)(oy + ly) * W + (ox + lx);
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

int launch_raster_fwd(gs_ctx* ctx, cudaStream_t s, float* rgb, float* depth, float* alpha) {
  const int units = ctx->cam.tiles_x * ctx->cam.tiles_y * 8;
  if (units == 0) return GS_OK;
  raster_fwd_kernel<false><<<units, 32, 0, s>>>(ctx->cam.W, ctx->cam.H, ctx->cam.tiles_x, ctx->tile_order, ctx->ranges,
                                                ctx->vals[ctx->sorted_buf], ctx->feat, ctx->bg[0], ctx->bg[1], ctx->bg[2],
                                                rgb, depth, alpha, ctx->final_T, ctx->n_contrib, nullptr);
  GS_LAUNCH_CHECK("raster_fwd_kernel");
  return GS_OK;
}

// Workload statistics of the forward (introspection only): re-walks every region's list with the forward's decisions.
int launch_workload_stats(gs_ctx* ctx, cudaStream_t s, uint64_t* out_host) {
  const int units = ctx->cam.tiles_x * ctx->cam.tiles_y * 8;
  if (!ctx->stats_ws) GS_CUDA(cudaMalloc((void**)&ctx->stats_ws, 8 * sizeof(unsigned long long)));
  unsigned long long* d = ctx->stats_ws;
  GS_CUDA(cudaMemsetAsync(d, 0, 8 * sizeof(unsigned long long), s));
  if (units > 0) {
    raster_fwd_kernel<true><<<units, 32, 0, s>>>(ctx->cam.W, ctx->cam.H, ctx->cam.tiles_x, ctx->tile_order, ctx->ranges,
                                                 ctx->vals[ctx->sorted_buf], ctx->feat, 0.f, 0.f, 0.f, nullptr, nullptr,
                                                 nullptr, nullptr, nullptr, d);
    GS_LAUNCH_CHECK("raster_fwd_kernel<stats>");
  }
  GS_CUDA(cudaMemcpyAsync(out_host, d, GS_NUM_WORKLOAD * sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
  GS_CUDA(cudaStreamSynchronize(s));
  return GS_OK;
}

}  // namespace gs

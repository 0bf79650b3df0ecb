// gs_raster.cu -- steps a6 (front-to-back compositing) and a8 (back-to-front per-pixel backward, reduced at warp
// level before global atomics).
//
// v2 design (evidence: profiles/r1_v1_baseline.md -- the one-pixel-per-thread kernels were bound by the LSU pipe:
// shuffles of the 10-value reduction and broadcast LDS of the Gaussian records):
//   * one WARP per tile region, 2 x NY interleaved pixels per lane (NY = 4: the whole 16x16 tile, NY = 2: half of it);
//     the Gaussian record is read from shared memory once per (region, Gaussian) instead of once per 32 pixels and
//     the conic products are shared across the lane's rows / columns;
//   * warps are autonomous (single-warp CTAs): no __syncthreads, early exit per region, hardware CTA scheduling
//     balances the very uneven tile lists;
//   * Gaussian records are gathered by cp.async (LDGSTS) into a double-buffered warp-private staging area, one batch
//     ahead of the compute, the sorted ids two batches ahead;
//   * phase 1 of every batch: lane g tests Gaussian g against the region (exact maximum of the concave power over the
//     region rectangle) -- Gaussians whose ellipse misses the region never reach the pixel loop;
//   * phase 2: the surviving Gaussians are taken FOUR at a time: 4 x NS powers evaluated together (ILP; the serial
//     latency per list entry is what bounds the longest tiles), one REDUX.OR over the packed slot masks;
//   * the alpha >= 1/255 test is taken in the power domain (power2 >= thr), so rejected pairs cost no MUFU;
//   * backward: the 10 per-Gaussian sums are accumulated over the lane's pixels first, then ONE 16-slot butterfly
//     reduce-scatter (16 SHFL) per (region, Gaussian) and one coalesced 10-lane RED.
#include "gs_internal.cuh"
#include "gs_raster.cuh"

namespace gs {

template <int NX, int NY, bool STATS>
__global__ void __launch_bounds__(32)
raster_fwd_kernel(int W, int H, int tiles_x, const uint32_t* __restrict__ order, const uint2* __restrict__ ranges, const uint32_t* __restrict__ ids,
                  const float4* __restrict__ feat, float bg0, float bg1, float bg2, float* __restrict__ rgb,
                  float* __restrict__ depth, float* __restrict__ alpha_out, float* __restrict__ final_T,
                  uint32_t* __restrict__ n_contrib, unsigned long long* __restrict__ stats) {
  constexpr int NS = NX * NY, RX = 2 / NX, RPT = RX * (4 / NY);  // slots per lane, regions per tile
  __shared__ __align__(16) float4 s_feat[2][kWarpBatch * 3];          // raw records, double-buffered (cp.async)
  __shared__ __align__(16) float4 s_rel[(kWarpBatch + kGroup) * 3];    // decoded records of the relevant Gaussians
  const int lane = threadIdx.x;
  const int tile = (int)__ldg(order + blockIdx.x / RPT), sub = blockIdx.x % RPT;
  const int ox = (tile % tiles_x) * GS_TILE + (sub % RX) * (8 * NX), oy = (tile / tiles_x) * GS_TILE + (sub / RX) * (4 * NY);
  const int lx = lane & 7, ly = lane >> 3;
  const float fx0 = (float)lx, fy0 = (float)ly;
  unsigned alive = 0;
#pragma unroll
  for (int k = 0; k < NS; ++k)
    if (ox + lx + 8 * (k % NX) < W && oy + ly + 4 * (k / NX) < H) alive |= 1u << k;
  const unsigned inside = alive;
  const uint2 range = ranges[tile];
  const int n = (int)(range.y - range.x);
  const int nb = (n + kWarpBatch - 1) / kWarpBatch;
  float T[NS], C0[NS], C1[NS], C2[NS], D[NS];
  uint32_t last[NS];
#pragma unroll
  for (int k = 0; k < NS; ++k) { T[k] = 1.f; C0[k] = C1[k] = C2[k] = D[k] = 0.f; last[k] = 0; }
  unsigned long long n_eval = 0, n_blend = 0;

  auto issue = [&](int b, uint32_t id) {
    if (b * kWarpBatch + lane < n) {
      const float4* src = feat + 3 * (size_t)(id >> 8);  // list entries are index << 8 | region mask
      float4* dst = &s_feat[b & 1][lane * 3];
      cp_async16(dst, src); cp_async16(dst + 1, src + 1); cp_async16(dst + 2, src + 2);
    }
    cp_async_commit();
  };
  uint32_t id_next = 0;
  if (nb > 0) {
    issue(0, lane < n ? __ldg(ids + range.x + lane) : 0u);
    if (nb > 1) id_next = (kWarpBatch + lane < n) ? __ldg(ids + range.x + kWarpBatch + lane) : 0u;
  }
  bool stop = !__any_sync(kFull, alive != 0);
  for (int b = 0; b < nb && !stop; ++b) {
    if (b + 1 < nb) {
      issue(b + 1, id_next);
      const int i2 = (b + 2) * kWarpBatch + lane;
      if (b + 2 < nb) id_next = (i2 < n) ? __ldg(ids + range.x + i2) : 0u;
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncwarp();
    const int cnt = min(kWarpBatch, n - b * kWarpBatch);
    const float4* sf = s_feat[b & 1];
    // phase 1: which Gaussians of the batch can reach this region at all?  Lane g decodes Gaussian g once (region-local
    // mean) and, if relevant, appends the decoded record to the compact list s_rel in list order.
    bool relevant = false;
    float4 c0 = make_float4(0.f, 0.f, 0.f, 0.f), c1 = c0;
    if (lane < cnt) {
      GaussReg g;
      decode_gauss(sf[3 * lane], sf[3 * lane + 1], ox, oy, g);
      relevant = region_max_power(g, (float)(8 * NX - 1), (float)(4 * NY - 1)) >= g.thr - 1e-3f;
      c0 = make_float4(g.mx, g.my, g.A, g.B);
      c1 = make_float4(g.C, g.o, g.thr, __int_as_float(lane));
    }
    const unsigned rel = __ballot_sync(kFull, relevant);
    const int nrel = __popc(rel);
    if (relevant) {
      const int r = __popc(rel & ((1u << lane) - 1u));
      s_rel[3 * r] = c0; s_rel[3 * r + 1] = c1; s_rel[3 * r + 2] = sf[3 * lane + 2];
    }
    if (lane < kGroup) {  // padding records never pass: p >= NaN is false
      s_rel[3 * (nrel + lane)] = make_float4(0.f, 0.f, 0.f, 0.f);
      s_rel[3 * (nrel + lane) + 1] = make_float4(0.f, 0.f, __int_as_float(0x7fc00000), 0.f);
    }
    __syncwarp();
    // phase 2: front to back, four list entries at a time
    for (int r0 = 0; r0 < nrel; r0 += kGroup) {
      int jj[kGroup];
      GaussReg g[kGroup];
      float dx[kGroup][NX], dy[kGroup][NY], p[kGroup][NS];
      unsigned m = 0;
#pragma unroll
      for (int q = 0; q < kGroup; ++q) {
        const float4 a0 = s_rel[3 * (r0 + q)], a1 = s_rel[3 * (r0 + q) + 1];
        g[q].mx = a0.x; g[q].my = a0.y; g[q].A = a0.z; g[q].B = a0.w;
        g[q].C = a1.x; g[q].o = a1.y; g[q].thr = a1.z;
        jj[q] = __float_as_int(a1.w);
        eval_power<NX, NY>(g[q], fx0, fy0, dx[q], dy[q], p[q]);
#pragma unroll
        for (int k = 0; k < NS; ++k) m |= (p[q][k] >= g[q].thr) ? (1u << (q * NS + k)) : 0u;
      }
      if (STATS) {
#pragma unroll
        for (int q = 0; q < kGroup; ++q) n_eval += (r0 + q < nrel) ? __popc(alive) : 0;
      }
      constexpr unsigned kRep = 1u | (1u << NS) | (1u << (2 * NS)) | (1u << (3 * NS));  // replicate the slot mask over the group
      const unsigned any = __reduce_or_sync(kFull, m & (alive * kRep));
      if (any == 0) continue;
#pragma unroll
      for (int q = 0; q < kGroup; ++q) {
        if (((any >> (q * NS)) & ((1u << NS) - 1)) == 0) continue;
        const float4 f2 = s_rel[3 * (r0 + q) + 2];
        const unsigned mq = (m >> (q * NS)) & alive;
#pragma unroll
        for (int k = 0; k < NS; ++k) {
          if (any & (1u << (q * NS + k))) {
            if (mq & (1u << k)) {
              const float a = fminf(GS_ALPHA_MAX, __fmul_rn(g[q].o, ex2_approx(p[q][k])));
              if (T[k] < GS_T_MIN) {
                alive &= ~(1u << k);
              } else {
                const float w = a * T[k];
                C0[k] = fmaf(f2.x, w, C0[k]);
                C1[k] = fmaf(f2.y, w, C1[k]);
                C2[k] = fmaf(f2.z, w, C2[k]);
                D[k] = fmaf(f2.w, w, D[k]);
                T[k] = T[k] * (1.f - a);
                last[k] = (uint32_t)(b * kWarpBatch + jj[q] + 1);
                if (STATS) ++n_blend;
              }
            }
          }
        }
      }
      if (!__any_sync(kFull, alive != 0)) { stop = true; break; }
    }
    __syncwarp();
  }
  cp_async_wait<0>();
  const size_t HW = (size_t)W * H;
#pragma unroll
  for (int k = 0; k < NS; ++k) {
    if (inside & (1u << k)) {
      const size_t p = (size_t)(oy + ly + 4 * (k / NX)) * W + (ox + lx + 8 * (k % NX));
      if (!STATS) {
        if (rgb) {
          rgb[p] = fmaf(T[k], bg0, C0[k]);
          rgb[HW + p] = fmaf(T[k], bg1, C1[k]);
          rgb[2 * HW + p] = fmaf(T[k], bg2, C2[k]);
        }
        if (depth) depth[p] = D[k];
        if (alpha_out) alpha_out[p] = 1.f - T[k];
        final_T[p] = T[k];
        n_contrib[p] = last[k];
      }
    }
  }
  if (STATS) {
    unsigned long long v[4] = {n_eval, n_blend, 0ull, (unsigned long long)n * __popc(inside)};
#pragma unroll
    for (int k = 0; k < NS; ++k) v[2] += (inside & (1u << k)) ? last[k] : 0u;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) v[q] += __shfl_xor_sync(kFull, v[q], d);
      if (lane == 0 && v[q]) atomicAdd(stats + q, v[q]);
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Forward, 8x4-pixel regions, one pixel per lane (the default).  Evidence: profiles/r1_v3_regions.md -- the generic
// kernel above spent 57 warp instructions per relevant (region, Gaussian) entry, a third of them on the mask / vote /
// branch bookkeeping of its groups of four.  Here phase 2 is branch-free: every relevant entry is evaluated and blended
// under a per-lane predicate (alpha_eff = 0 where the pixel is not hit), four entries unrolled for ILP, one vote per
// four entries for the early exit.  ~26 instructions per entry.
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32)
raster_fwd84_kernel(int W, int H, int tiles_x, const uint32_t* __restrict__ order, const uint2* __restrict__ ranges,
                    const uint32_t* __restrict__ ids, const float4* __restrict__ feat, float bg0, float bg1, float bg2,
                    float* __restrict__ rgb, float* __restrict__ depth, float* __restrict__ alpha_out,
                    float* __restrict__ final_T, uint32_t* __restrict__ n_contrib) {
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

  // phase 1: the list entries are (index << 8 | region mask) -- gs_bin_tiles already decided which regions of the tile
  // a Gaussian can reach.  Lane g looks at entry g of the batch; the relevant ones are compacted (ballot rank) and only
  // their records are staged, one batch ahead.
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
    if (lane < nrel) {  // decode once per (region, Gaussian), in place: region-local mean
      GaussReg g;
      decode_gauss(sf[3 * lane], sf[3 * lane + 1], ox, oy, g);
      sf[3 * lane] = make_float4(g.mx, g.my, g.A, g.B);
      sf[3 * lane + 1] = make_float4(g.C, g.o, g.thr, __uint_as_float(s_pos[b & 1][lane]));
    }
    if (lane < kGroup) {  // padding records never pass: p >= NaN is false
      sf[3 * (nrel + lane)] = make_float4(0.f, 0.f, 0.f, 0.f);
      sf[3 * (nrel + lane) + 1] = make_float4(0.f, 0.f, __int_as_float(0x7fc00000), 0.f);
      sf[3 * (nrel + lane) + 2] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    __syncwarp();
    // phase 2: front to back, branch-free
    for (int r0 = 0; r0 < nrel; r0 += kGroup) {
#pragma unroll
      for (int q = 0; q < kGroup; ++q) {
        const float4 a0 = sf[3 * (r0 + q)], a1 = sf[3 * (r0 + q) + 1], f2 = sf[3 * (r0 + q) + 2];
        float dx, dy;
        const float p = eval_power1(a0.x, a0.y, a0.z, a0.w, a1.x, fx0, fy0, dx, dy);
        const bool hit = (p >= a1.z) && (T >= GS_T_MIN);   // alpha >= 1/255 and the pixel has not terminated
        const float a = hit ? fminf(GS_ALPHA_MAX, __fmul_rn(a1.y, ex2_approx(p))) : 0.f;
        const float w = a * T;
        C0 = fmaf(f2.x, w, C0);
        C1 = fmaf(f2.y, w, C1);
        C2 = fmaf(f2.z, w, C2);
        D = fmaf(f2.w, w, D);
        T = T * (1.f - a);
        last = hit ? __float_as_uint(a1.w) : last;
      }
      if (!__any_sync(kFull, T >= GS_T_MIN)) { stop = true; break; }
    }
    __syncwarp();
  }
  cp_async_wait<0>();
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

static int launch_fwd84(gs_ctx* ctx, cudaStream_t s, float* rgb, float* depth, float* alpha) {
  const int units = ctx->cam.tiles_x * ctx->cam.tiles_y * 8;
  raster_fwd84_kernel<<<units, 32, 0, s>>>(ctx->cam.W, ctx->cam.H, ctx->cam.tiles_x, ctx->tile_order, ctx->ranges,
                                           ctx->vals[ctx->sorted_buf], ctx->feat, ctx->bg[0], ctx->bg[1], ctx->bg[2],
                                           rgb, depth, alpha, ctx->final_T, ctx->n_contrib);
  GS_LAUNCH_CHECK("raster_fwd84_kernel");
  return GS_OK;
}

template <int NX, int NY>
static int launch_fwd_t(gs_ctx* ctx, cudaStream_t s, float* rgb, float* depth, float* alpha) {
  const int units = ctx->cam.tiles_x * ctx->cam.tiles_y * (2 / NX) * (4 / NY);
  raster_fwd_kernel<NX, NY, false><<<units, 32, 0, s>>>(ctx->cam.W, ctx->cam.H, ctx->cam.tiles_x, ctx->tile_order,
                                                         ctx->ranges, ctx->vals[ctx->sorted_buf], ctx->feat,
                                                         ctx->bg[0], ctx->bg[1], ctx->bg[2], rgb, depth, alpha,
                                                         ctx->final_T, ctx->n_contrib, nullptr);
  GS_LAUNCH_CHECK("raster_fwd_kernel");
  return GS_OK;
}

// region shape per warp = (8 NX) x (4 NY) pixels; selectable for tuning (GS_RASTER_FWD / GS_RASTER_BWD = "NXNY")
#define GS_DISPATCH(shape, F, ...)                      \
  switch (shape) {                                      \
    case 11: return F<1, 1>(__VA_ARGS__);               \
    case 12: return F<1, 2>(__VA_ARGS__);               \
    case 21: return F<2, 1>(__VA_ARGS__);               \
    case 22: return F<2, 2>(__VA_ARGS__);               \
    default: return F<2, 4>(__VA_ARGS__);               \
  }

int launch_raster_fwd(gs_ctx* ctx, cudaStream_t s, float* rgb, float* depth, float* alpha) {
  if (ctx->cam.tiles_x * ctx->cam.tiles_y == 0) return GS_OK;
  if (ctx->shape_fwd == 0) return launch_fwd84(ctx, s, rgb, depth, alpha);
  GS_DISPATCH(ctx->shape_fwd, launch_fwd_t, ctx, s, rgb, depth, alpha)
}

// Workload statistics of the forward (introspection only): re-walks every pixel's list with the forward's decisions.
int launch_workload_stats(gs_ctx* ctx, cudaStream_t s, uint64_t* out_host) {
  const int tiles = ctx->cam.tiles_x * ctx->cam.tiles_y;
  if (!ctx->stats_ws) GS_CUDA(cudaMalloc((void**)&ctx->stats_ws, 8 * sizeof(unsigned long long)));
  unsigned long long* d = ctx->stats_ws;
  GS_CUDA(cudaMemsetAsync(d, 0, 4 * sizeof(unsigned long long), s));
  if (tiles > 0) {
    raster_fwd_kernel<2, 4, true><<<tiles, 32, 0, s>>>(ctx->cam.W, ctx->cam.H, ctx->cam.tiles_x, ctx->tile_order,
                                                        ctx->ranges, ctx->vals[ctx->sorted_buf], ctx->feat, 0.f, 0.f,
                                                        0.f, nullptr, nullptr, nullptr, nullptr, nullptr, d);
    GS_LAUNCH_CHECK("raster_fwd_kernel<stats>");
  }
  GS_CUDA(cudaMemcpyAsync(out_host, d, 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
  GS_CUDA(cudaStreamSynchronize(s));
  return GS_OK;
}

}  // namespace gs

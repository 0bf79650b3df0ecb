// gs_raster.cu -- step a6: per-tile front-to-back compositing (oracle reading C1 step 7).
//
// Design as built (v10; history and evidence: profiles/r1_*.md, r2_v7_tile_cta.md, r2_v9_ring.md, r2_v10_chain.md).  Up to
// round-2 v6 every 8x4 region was an autonomous single-warp CTA that gathered, decoded and compacted its own records: per
// relevant (region, Gaussian) entry the forward spent 47 warp instructions and 13.8 shared-memory wavefronts, of which
// only ~22 / 7.4 were the blend itself.  Now:
//   * one CTA of FOUR warps per HALF tile (GS_FWD_WARPS = 4; two CTAs per 16x16 tile), a warp = one 8x4-pixel region, one
//     pixel per lane; tiles are visited in the longest-list-first order gs_bin_tiles wrote (`order`);
//   * the tile's list is staged in rounds of 128 entries (GS_FWD_BATCH) into a ring of 4 stages with 2 rounds of slack
//     (GS_FWD_RING_STAGES / _DELAY, Ring<> in gs_raster.cuh): every thread is a producer -- one 16-byte cp.async.cg for
//     the instance record {u0, v0, list word} and two for the 32 contiguous bytes {l11, l21, l22, lo}{r, g, b, z} of the
//     Gaussian, gathered by visible slot -- and signals the stage's `full` mbarrier through cp.async.mbarrier.arrive;
//     a warp releases a stage through its `empty` mbarrier.  There is NO block-wide barrier in the loop: the four warps
//     drift up to kDelay + 1 rounds apart; staging stops when no warp of the CTA has a live pixel (s_live);
//   * every warp turns the round's 128 region masks into a list of byte offsets of the entries relevant to ITS region
//     (ballots, ranks by popc, 16-bit stores into s_idx) and walks that list front to back, four entries per step
//     (kGroup): the records are read as broadcast LDS.128 x 2 + LDS.64;
//   * the pixel loop is branch-free: every relevant entry is evaluated and blended under a per-lane predicate (alpha_eff
//     = 0 where the pixel is not hit or has terminated); alpha >= 1/255 is tested in the exponent domain against a
//     constant, so rejected pairs cost no MUFU and the opacity never enters the loop.
#include "gs_internal.cuh"
#include "gs_raster.cuh"

namespace gs {

// NW: warps (= regions) per CTA.  8: one CTA per tile; 4 / 2: half / quarter tiles -- the list is then staged 2 / 4 times
// per tile (profiles/r2_v7_tile_cta.md, r2_v9_ring.md).
#ifndef GS_FWD_WARPS
#define GS_FWD_WARPS 4
#endif
#ifndef GS_FWD_RING_STAGES
#define GS_FWD_RING_STAGES 4
#endif
#ifndef GS_FWD_RING_DELAY
#define GS_FWD_RING_DELAY 2
#endif
#ifndef GS_FWD_BATCH
#define GS_FWD_BATCH 128
#endif
constexpr int kTileBatch = GS_FWD_BATCH, kPadIdx = kTileBatch;  // list entries staged per round by a CTA; padding record
constexpr int kStages = GS_FWD_RING_STAGES, kDelay = GS_FWD_RING_DELAY, kAhead = kStages - kDelay;  // gs_raster.cuh
static_assert(kDelay >= 0 && kAhead >= 2, "ring shape");

// STATS = true: the same walk with the same decisions, counting the workload instead of writing the image
// (gs_get_workload; never on the timed path).
template <int NW, bool STATS>
__global__ void __launch_bounds__(NW * 32)
raster_fwd_kernel(int W, int H, int tiles_x, const uint32_t* __restrict__ order, const uint2* __restrict__ ranges,
                  const float4* __restrict__ inst, const float4* __restrict__ feat,
                  float bg0, float bg1, float bg2, float* __restrict__ rgb, float* __restrict__ depth,
                  float* __restrict__ alpha_out, float* __restrict__ final_T, uint32_t* __restrict__ n_contrib,
                  unsigned long long* __restrict__ stats) {
  constexpr int CPT = 8 / NW;  // CTAs per tile
  constexpr int TPE = Ring<NW, kStages, kTileBatch>::TPE;
  __shared__ __align__(16) Ring<NW, kStages, kTileBatch> ring;
  // per warp: byte offsets (into the stage) of the round's relevant entries, in list order
  __shared__ __align__(8) uint16_t s_idx[NW][kTileBatch + kGroup];
  __shared__ int s_live;  // warps of the CTA that still have a live pixel: staging stops when it reaches zero
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  pdl_enter();
  const int tile = (int)__ldg(order + blockIdx.x / CPT), sub = (blockIdx.x % CPT) * NW + warp;
  const int tx0 = (tile % tiles_x) * GS_TILE, ty0 = (tile / tiles_x) * GS_TILE;
  const int X = (sub % 2) * 8 + (lane & 7), Y = (sub / 2) * 4 + (lane >> 3);  // tile-local pixel of this lane
  const float fx0 = (float)X, fy0 = (float)Y;
  const bool inside = tx0 + X < W && ty0 + Y < H;
  const uint2 range = ranges[tile];
  const int n = (int)(range.y - range.x);
  const int nb = (n + kTileBatch - 1) / kTileBatch;
  // T starts at 0 for a lane outside the image, so such a lane never blends (and writes nothing)
  float T = inside ? 1.f : 0.f, C0 = 0.f, C1 = 0.f, C2 = 0.f, D = 0.f;
  uint32_t last48 = 0;                // 48 x (list position + 1) of the last blended entry
  unsigned long long n_eval = 0, n_blend = 0;
  uint32_t rank = 0, last_rank = 0;   // STATS: relevant entries walked so far; rank of the pixel's last blended one

  bool alive_warp = __any_sync(kFull, inside);
  ring.init(tid);
  if (tid == 0) s_live = 0;
  __syncthreads();
  if (lane == 0 && alive_warp) atomicAdd(&s_live, 1);
  // producer state: this thread stages entry e_pro of every round; the list word is fetched one step ahead
  const int e_pro = tid / TPE;
  uint32_t v_pre = 0;
  auto fetch = [&](int k) {
    const int i = k * kTileBatch + e_pro;
    v_pre = i < n ? __float_as_uint(__ldg(&inst[range.x + i].z)) : 0u;
  };
  fetch(0);
#pragma unroll
  for (int k = 0; k < kAhead; ++k) {
    if (k < nb) ring.produce(k, k * kTileBatch + e_pro, n, range.x, v_pre, tid, inst, feat);
    fetch(k + 1);
  }
  __syncthreads();  // s_live is complete
  const volatile int* live = &s_live;
  uint32_t base48 = 48u;  // 48 x (list position + 1) of entry 0 of the round
  for (int j = 0; j < nb; ++j, base48 += 48u * kTileBatch) {
    const int stage = j & (kStages - 1);
    if (alive_warp) {
      mbar_wait(&ring.full[stage], (uint32_t)(j / kStages) & 1u);
      const StageBuf<kTileBatch>& sb = ring.st[stage];
      // the entries of this round that can reach this warp's region, as a list of byte offsets in list order
      const int left = n - j * kTileBatch;  // entries of the round that exist (what lies beyond is stale)
      constexpr int NCH = kTileBatch / 32;
      bool rr[NCH];
      unsigned bb[NCH];
      int nrel = 0;
#pragma unroll
      for (int c = 0; c < NCH; ++c) {
        rr[c] = ((sb.rec[lane + 32 * c].ent >> sub) & 1u) && lane + 32 * c < left;
        bb[c] = __ballot_sync(kFull, rr[c]);
        nrel += __popc(bb[c]);
      }
      if (nrel) {
        const unsigned lt = (1u << lane) - 1u;
        uint16_t* idx = s_idx[warp];
        int at = 0;
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
          if (rr[c]) idx[at + __popc(bb[c] & lt)] = (uint16_t)((lane + 32 * c) * 48);
          at += __popc(bb[c]);
        }
        if (lane < kGroup) idx[nrel + lane] = (uint16_t)(kPadIdx * 48);
        __syncwarp();
        const char* recs = reinterpret_cast<const char*>(sb.rec);
        for (int r = 0; r < nrel; r += kGroup) {
          const uint2 o4 = *reinterpret_cast<const uint2*>(idx + r);
          const uint32_t off[kGroup] = {o4.x & 0xffffu, o4.x >> 16, o4.y & 0xffffu, o4.y >> 16};
#pragma unroll
          for (int q = 0; q < kGroup; ++q) {
            const StageRec& e = *reinterpret_cast<const StageRec*>(recs + off[q]);
            const float4 a0 = e.g, f2 = e.c;
            const float2 uv = e.uv;
            const float p = eval_power(uv.x, uv.y, a0.x, a0.y, a0.z, a0.w, fx0, fy0);
            const bool alive = T >= GS_T_MIN;
            const bool hit = (p >= GS_POWER_MIN) && alive;   // alpha >= 1/255 and the pixel has not terminated
            const float a = hit ? fminf(GS_ALPHA_MAX, ex2_approx(p)) : 0.f;
            const float w = a * T;
            C0 = fmaf(f2.x, w, C0);
            C1 = fmaf(f2.y, w, C1);
            C2 = fmaf(f2.z, w, C2);
            D = fmaf(f2.w, w, D);
            T = fmaf(-a, T, T);
            last48 = hit ? base48 + off[q] : last48;
            if (STATS && r + q < nrel) {
              ++rank;
              n_eval += alive ? 1 : 0;
              n_blend += hit ? 1 : 0;
              last_rank = hit ? rank : last_rank;
            }
          }
          if (!__any_sync(kFull, T >= GS_T_MIN)) { alive_warp = false; break; }
        }
        if (!alive_warp && lane == 0) atomicSub(&s_live, 1);
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&ring.empty[stage]);  // this warp is done with the stage (a dead warp: at once)
    // refill: the stage of round j - kDelay takes round j + kAhead once every warp has released it
    const int k = j + kAhead;
    if (k < nb) {
      bool stop = false;
      if (j >= kDelay) {
        const uint32_t par = (uint32_t)((j - kDelay) / kStages) & 1u;
        while (!mbar_try_wait(&ring.empty[k & (kStages - 1)], par))
          if (*live == 0) { stop = true; break; }   // the warps this one waits for have left
      }
      if (stop) break;
      ring.produce(k, k * kTileBatch + e_pro, n, range.x, v_pre, tid, inst, feat);
      fetch(k + 1);
    }
    if (*live == 0) break;  // no pixel of the CTA is alive any more
  }
  cp_async_wait_all();
  const uint32_t last = last48 / 48u;
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
    const size_t p = (size_t)(ty0 + Y) * W + (tx0 + X);
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
  const int tiles = ctx->cam.tiles_x * ctx->cam.tiles_y;
  if (tiles == 0) return GS_OK;
  constexpr int NW = GS_FWD_WARPS;
  GS_LAUNCH_PDL((raster_fwd_kernel<NW, false>), tiles * (8 / NW), NW * 32, 0, s, ctx->cam.W, ctx->cam.H, ctx->cam.tiles_x,
                (const uint32_t*)ctx->tile_order, (const uint2*)ctx->ranges, (const float4*)ctx->inst_rec, (const float4*)ctx->feat, ctx->bg[0], ctx->bg[1], ctx->bg[2], rgb, depth, alpha,
                ctx->final_T, ctx->n_contrib, (unsigned long long*)nullptr);
  GS_LAUNCH_CHECK("raster_fwd_kernel");
  return GS_OK;
}

// Workload statistics of the forward (introspection only): re-walks every tile's list with the forward's decisions.
int launch_workload_stats(gs_ctx* ctx, cudaStream_t s, uint64_t* out_host) {
  const int tiles = ctx->cam.tiles_x * ctx->cam.tiles_y;
  if (!ctx->stats_ws) GS_CUDA(cudaMalloc((void**)&ctx->stats_ws, 8 * sizeof(unsigned long long)));
  unsigned long long* d = ctx->stats_ws;
  GS_CUDA(cudaMemsetAsync(d, 0, 8 * sizeof(unsigned long long), s));
  if (tiles > 0) {
    raster_fwd_kernel<8, true><<<tiles, 256, 0, s>>>(ctx->cam.W, ctx->cam.H, ctx->cam.tiles_x, ctx->tile_order, ctx->ranges,
                                                     ctx->inst_rec, ctx->feat, 0.f, 0.f, 0.f,
                                                     nullptr, nullptr, nullptr, nullptr, nullptr, d);
    GS_LAUNCH_CHECK("raster_fwd_kernel<stats>");
  }
  GS_CUDA(cudaMemcpyAsync(out_host, d, GS_NUM_WORKLOAD * sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
  GS_CUDA(cudaStreamSynchronize(s));
  return GS_OK;
}

}  // namespace gs

// gs_raster_bwd.cu -- step a8: back-to-front per-pixel backward of the compositing, reduced per (region, Gaussian)
// before global atomics.
//
// v4 design (evidence: profiles/r1_v3_regions.md -- one warp per 8x4-pixel region, one pixel per lane; the register
// butterfly that reduced the 10 per-Gaussian sums over the lanes was 42 % of the instructions, and parking the 10
// values per lane in shared memory instead made the kernel LSU-bound: 20 wavefronts per (region, Gaussian)):
//   * PIXEL phase (lane = pixel): walks the region's list back to front exactly like the forward walks it front to
//     back (cp.async staging, phase-1 rectangle culling, groups of four), rebuilds T, and for every Gaussian that
//     reaches at least one pixel hands over just TWO numbers per lane -- gp = alpha dL/dalpha (0 where clamped or not
//     blended) and w = alpha T -- with one STS.64 into a [slot][pixel] table;
//   * GAUSSIAN phase (lane = Gaussian slot x half of the region), run when 16 slots are full: every lane walks 16
//     pixels of ITS Gaussian, re-forms the WHITENED offsets (u, v) = L^T (pixel - mean) from the slot's record
//     (gs_raster.cuh: |u|, |v| <= ~4 wherever gp != 0) and accumulates the 10 sums (moments of gp in (u, v); w-weighted
//     upstream colour / depth gradients) in registers -- no cross-lane reduction except one SHFL per sum to join the
//     two halves -- and the 16 x 10 totals leave through shared memory as coalesced RED.ADD.F32.  Moments in the
//     whitened frame are well conditioned for any footprint: dL/dSigma' = L M2 L^T / (2 k^2) needs no cancellation
//     (moments of dx, dy lost 3 digits on 1000:1 footprints through -Q gQ Q).
//   ~15 instructions and ~5 shared-memory wavefronts per (region, Gaussian) for the whole reduction.
#include "gs_internal.cuh"
#include "gs_raster.cuh"

namespace gs {

#ifndef GS_BWD_MIN_BLOCKS
#define GS_BWD_MIN_BLOCKS 22
#endif
constexpr int kSlots = 16;     // Gaussians per flush of the Gaussian phase
constexpr int kPairRow = 33;   // float2 per slot row (32 pixels + 1: conflict-free transposed LDS.64)
constexpr int kOutVals = 10;   // sums per Gaussian (gs_internal.cuh kG2D, first 10)

// Gaussian phase.  SPLIT = 2: lane = (slot = lane & 15, half = lane >> 4), 2 pixel rows per lane;
//                  SPLIT = 4: lane = (slot = lane & 7, quarter = lane >> 3), 1 pixel row per lane (tail flush, <= 8 slots).
// Record of the Gaussian in slot (lane & 15), kept in registers between the pixel phase and the flush: the whitened
// offset of the region origin and the visible slot; L is re-read from the feature record at the flush (one LDG.128 per
// lane per 16 Gaussians) instead of being carried in three more registers (80 registers is the occupancy limit here).
struct SlotRec { float u0, v0; };

template <int SPLIT>
__device__ __forceinline__ void gaussian_phase(float2* s_pair, const float4* s_pix, int nslot, int lane, const SlotRec& sr,
                                               uint32_t slot_id, const float4* __restrict__ feat, float* __restrict__ g2d) {
  constexpr int LS = 32 / SPLIT, R = 4 / SPLIT;  // slots per pass, pixel rows per lane
  __syncwarp();
  const int slot = lane & (LS - 1), part = lane / LS;
  // the slot records live in registers: lane s (and lane s + 16) holds the record of slot s
  float u0 = sr.u0, v0 = sr.v0;
  uint32_t id = slot_id;
  if (SPLIT == 4) {
    u0 = __shfl_sync(kFull, sr.u0, slot); v0 = __shfl_sync(kFull, sr.v0, slot);
    id = __shfl_sync(kFull, slot_id, slot);
  }
  float4 L = make_float4(0.f, 0.f, 0.f, 0.f);
  if (slot < nslot) L = __ldg(feat + 3 * (size_t)id + 1);  // l11, l21, l22
  struct { float u0, v0, l11, l21, l22; } g = {u0, v0, L.x, L.y, L.z};
  float ub[R], vs[R];
#pragma unroll
  for (int r = 0; r < R; ++r) {
    const float y = (float)(part * R + r);
    ub[r] = fmaf(g.l21, y, g.u0);
    vs[r] = fmaf(g.l22, y, g.v0);
  }
  const float2* pr = s_pair + slot * kPairRow + part * (R * 8);
  const float4* px = s_pix + part * (R * 8);
  float acc[kOutVals];
#pragma unroll
  for (int u = 0; u < kOutVals; ++u) acc[u] = 0.f;
#pragma unroll
  for (int r = 0; r < R; ++r) {
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      const float2 pw = pr[r * 8 + c];  // gp, w of (this Gaussian, pixel)
      const float4 gu = px[r * 8 + c];  // upstream dL/dRGB, dL/dDepth of the pixel
      const float uu = fmaf(g.l11, (float)c, ub[r]);
      const float gx = pw.x * uu, gy = pw.x * vs[r];
      acc[0] += gx;
      acc[1] += gy;
      acc[2] = fmaf(gx, uu, acc[2]);
      acc[3] = fmaf(gx, vs[r], acc[3]);
      acc[4] = fmaf(gy, vs[r], acc[4]);
      acc[5] += pw.x;
      acc[6] = fmaf(pw.y, gu.x, acc[6]);
      acc[7] = fmaf(pw.y, gu.y, acc[7]);
      acc[8] = fmaf(pw.y, gu.z, acc[8]);
      acc[9] = fmaf(pw.y, gu.w, acc[9]);
    }
  }
#pragma unroll
  for (int u = 0; u < kOutVals; ++u) {
    acc[u] += __shfl_xor_sync(kFull, acc[u], 16);
    if (SPLIT == 4) acc[u] += __shfl_xor_sync(kFull, acc[u], 8);
  }
  // the totals leave through shared memory (the pair table is consumed: the shuffles above converged the warp) so that
  // consecutive lanes carry consecutive values of consecutive slots: coalesced RED
  float* s_out = reinterpret_cast<float*>(s_pair);
  if (part == 0) {
#pragma unroll
    for (int u = 0; u < kOutVals; ++u) s_out[slot * kOutVals + u] = acc[u];
  }
  __syncwarp();
  const int total = nslot * kOutVals;
#pragma unroll
  for (int t = 0; t < (LS * kOutVals + 31) / 32; ++t) {
    const int idx = t * 32 + lane;
    const int sl_i = min(idx / kOutVals, LS - 1), val = idx - sl_i * kOutVals;
    const uint32_t id = __shfl_sync(kFull, slot_id, sl_i);
    if (idx < total) atomicAdd(g2d + (size_t)id * kG2D + val, s_out[idx]);
  }
  __syncwarp();
}

template <bool HAS_GA>
__global__ void __launch_bounds__(32, GS_BWD_MIN_BLOCKS)
raster_bwd_kernel(int W, int H, int tiles_x, const uint32_t* __restrict__ order, const uint2* __restrict__ ranges,
                  const uint32_t* __restrict__ ids, const float4* __restrict__ feat, float bg0, float bg1, float bg2,
                  const float* __restrict__ final_T, const uint32_t* __restrict__ n_contrib,
                  const float* __restrict__ d_rgb, const float* __restrict__ d_depth, const float* __restrict__ d_alpha,
                  float* __restrict__ g2d) {
  constexpr int RPT = 8;  // 8x4-pixel regions per 16x16 tile
  __shared__ __align__(16) float4 s_feat[2][(kWarpBatch + kGroup) * 3];  // records of the relevant entries, decoded in place
  __shared__ uint32_t s_tag[2][kWarpBatch];
  __shared__ __align__(16) float2 s_pair[kSlots * kPairRow];
  __shared__ __align__(16) float4 s_pix[32];
  const int lane = threadIdx.x;
  const int tile = (int)__ldg(order + blockIdx.x / RPT), sub = blockIdx.x % RPT;
  const int ox = (tile % tiles_x) * GS_TILE + (sub % 2) * 8, oy = (tile / tiles_x) * GS_TILE + (sub / 2) * 4;
  const int lx = lane & 7, ly = lane >> 3;
  const float fx0 = (float)lx, fy0 = (float)ly;
  const uint2 range = ranges[tile];
  const size_t HW = (size_t)W * H;
  float T = 1.f, gC0 = 0.f, gC1 = 0.f, gC2 = 0.f, gD = 0.f, gA = 0.f;
  uint32_t last = 0;
  {
    const int X = ox + lx, Y = oy + ly;
    if (X < W && Y < H) {
      const size_t p = (size_t)Y * W + X;
      T = final_T[p];
      last = n_contrib[p];
      gC0 = d_rgb[p]; gC1 = d_rgb[HW + p]; gC2 = d_rgb[2 * HW + p];
      if (d_depth) gD = d_depth[p];
      if (HAS_GA) gA = d_alpha[p];
    }
  }
  s_pix[lane] = make_float4(gC0, gC1, gC2, gD);
  float S = T * (gC0 * bg0 + gC1 * bg1 + gC2 * bg2);
  const int n = (int)__reduce_max_sync(kFull, last);  // deepest blended list position of the region
  const int nb = (n + kWarpBatch - 1) / kWarpBatch;
  int nslot = 0;
  float2* pair_ptr = s_pair + lane;     // where this lane's (gp, w) of the next slot goes
  SlotRec slot = {0.f, 0.f};  // record of slot (lane & 15), kept in registers
  uint32_t slot_id = 0;

  // phase 1: the list entries are (index << 8 | region mask) -- gs_bin_tiles already decided which regions of the tile
  // a Gaussian can reach.  Lane g looks at entry g of the batch; the relevant ones are compacted in REVERSE list order
  // (ballot rank) and only their records are staged, one batch ahead; tag = index << 5 | position in the batch.
  auto issue = [&](int b, uint32_t v) -> int {
    const bool relevant = (b * kWarpBatch + lane < n) && ((v >> sub) & 1u);
    const unsigned rel = __ballot_sync(kFull, relevant);
    const int cnt = __popc(rel);
    if (relevant) {
      const int r = cnt - 1 - __popc(rel & ((1u << lane) - 1u));
      const float4* src = feat + 3 * (size_t)(v >> 8);
      float4* dst = &s_feat[b & 1][r * 3];
      cp_async16(dst, src); cp_async16(dst + 1, src + 1); cp_async16(dst + 2, src + 2);
      s_tag[b & 1][r] = ((v >> 8) << 5) | (uint32_t)lane;
    }
    cp_async_commit();
    return cnt;
  };
  uint32_t v_next = 0;
  int nrel = 0, nrel_next = 0;
  if (nb > 0) {
    const int i0 = (nb - 1) * kWarpBatch + lane;
    nrel_next = issue(nb - 1, i0 < n ? __ldg(ids + range.x + i0) : 0u);
    if (nb > 1) v_next = __ldg(ids + range.x + (nb - 2) * kWarpBatch + lane);
  }
  for (int b = nb - 1; b >= 0; --b) {
    nrel = nrel_next;
    if (b >= 1) {
      nrel_next = issue(b - 1, v_next);
      if (b >= 2) v_next = __ldg(ids + range.x + (b - 2) * kWarpBatch + lane);
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncwarp();
    if (nrel == 0) continue;
    const int lastb = (int)last - b * kWarpBatch;  // entries of this batch at positions < lastb were blended by this pixel
    float4* sf = s_feat[b & 1];
    if (lane < nrel) {  // decode once per (region, Gaussian), in place: whitened region-local record (gs_raster.cuh)
      const float4 f0 = sf[3 * lane], f1 = sf[3 * lane + 1];
      float u0, v0, mx, my;
      decode_whitened(f0, f1, ox, oy, u0, v0, mx, my);
      sf[3 * lane] = make_float4(u0, v0, f1.x, f1.y);
      sf[3 * lane + 1] = make_float4(f1.z, f0.w, __uint_as_float(s_tag[b & 1][lane]), 0.f);
    }
    if (lane < kGroup) {  // padding records never pass: lo = -inf  =>  p2 = -inf
      sf[3 * (nrel + lane)] = make_float4(0.f, 0.f, 0.f, 0.f);
      sf[3 * (nrel + lane) + 1] = make_float4(0.f, -INFINITY, 0.f, 0.f);
    }
    __syncwarp();
    for (int r0 = 0; r0 < nrel; r0 += kGroup) {  // back to front, four list entries at a time
      float4 a0[kGroup], a1[kGroup];
      float p[kGroup];
      bool hit[kGroup];
      unsigned bal[kGroup];
#pragma unroll
      for (int q = 0; q < kGroup; ++q) {
        a0[q] = sf[3 * (r0 + q)];      // u0, v0, l11, l21
        a1[q] = sf[3 * (r0 + q) + 1];  // l22, lo, tag
        p[q] = eval_power(a0[q].x, a0[q].y, a0[q].z, a0[q].w, a1[q].x, a1[q].y, fx0, fy0);
        // blended by the forward: alpha >= 1/255 and in front of the pixel's last contributor
        hit[q] = p[q] >= GS_POWER_MIN && (int)(__float_as_uint(a1[q].z) & 31u) < lastb;
        bal[q] = __ballot_sync(kFull, hit[q]);
      }
#pragma unroll
      for (int q = 0; q < kGroup; ++q) {
        if (bal[q] == 0) continue;  // the Gaussian reaches no pixel of the region
        float gp = 0.f, w = 0.f;
        if (hit[q]) {
          const float4 f2 = sf[3 * (r0 + q) + 2];
          const float og = ex2_approx(p[q]);  // opacity * G: log2(opacity) is folded into the exponent
          const float a = fminf(GS_ALPHA_MAX, og);
          const float ioma = rcp_approx(1.f - a);
          T *= ioma;  // transmittance in front of this Gaussian
          w = a * T;
          float wi = fmaf(gC0, f2.x, fmaf(gC1, f2.y, fmaf(gC2, f2.z, gD * f2.w)));
          if (HAS_GA) wi += gA;
          const float dalpha = fmaf(T, wi, -S * ioma);
          S = fmaf(wi, w, S);
          gp = (og <= GS_ALPHA_MAX) ? a * dalpha : 0.f;  // no gradient through the clamp (Q2)
        }
        *pair_ptr = make_float2(gp, w);
        pair_ptr += kPairRow;
        if ((lane & (kSlots - 1)) == nslot) {
          slot.u0 = a0[q].x; slot.v0 = a0[q].y;
          slot_id = __float_as_uint(a1[q].z) >> 5;
        }
        if (++nslot == kSlots) {
          gaussian_phase<2>(s_pair, s_pix, kSlots, lane, slot, slot_id, feat, g2d);
          nslot = 0;
          pair_ptr = s_pair + lane;
        }
      }
    }
    __syncwarp();
  }
  if (nslot > 8) gaussian_phase<2>(s_pair, s_pix, nslot, lane, slot, slot_id, feat, g2d);
  else if (nslot > 0) gaussian_phase<4>(s_pair, s_pix, nslot, lane, slot, slot_id, feat, g2d);
}

int launch_raster_bwd(gs_ctx* ctx, cudaStream_t s, const float* d_rgb, const float* d_depth, const float* d_alpha) {
  const int units = ctx->cam.tiles_x * ctx->cam.tiles_y * 8;
  if (units == 0) return GS_OK;
#define GS_BWD(GA)                                                                                                  \
  raster_bwd_kernel<GA><<<units, 32, 0, s>>>(ctx->cam.W, ctx->cam.H, ctx->cam.tiles_x, ctx->tile_order, ctx->ranges, \
                                             ctx->vals[ctx->sorted_buf], ctx->feat, ctx->bg[0], ctx->bg[1],         \
                                             ctx->bg[2], ctx->final_T, ctx->n_contrib, d_rgb, d_depth, d_alpha,     \
                                             ctx->g2d)
  if (d_alpha) GS_BWD(true); else GS_BWD(false);
#undef GS_BWD
  GS_LAUNCH_CHECK("raster_bwd_kernel");
  return GS_OK;
}

}  // namespace gs

// gs_raster_bwd.cu -- step a8: back-to-front per-pixel backward of the compositing, reduced per (region, Gaussian)
// before global atomics.
//
// Same structure as the forward (gs_raster.cu): one CTA of four warps per HALF tile, a warp = one 8x4-pixel region, the
// list staged in rounds of 128 entries (GS_BWD_BATCH) through the mbarrier / cp.async ring of gs_raster.cuh -- here two
// stages and no slack (GS_BWD_RING_STAGES = 2, _DELAY = 0: 12 KB; a deeper ring costs a CTA of occupancy), no block-wide
// barrier in the loop -- walked from the deepest blended position of the half tile back to the front.  Per warp (evidence: profiles/r1_v3_regions.md -- a register butterfly that
// reduced the 10 per-Gaussian sums over the lanes was 42 % of the instructions, and parking the 10 values per lane in
// shared memory made the kernel LSU-bound at 20 wavefronts per (region, Gaussian)):
//   * PIXEL phase (lane = pixel): walks the region's relevant entries back to front, rebuilds T, and for every Gaussian
//     that reaches at least one pixel hands over just TWO numbers per lane -- gp = alpha dL/dalpha (0 where clamped or not
//     blended) and w = alpha T -- with one STS.64 into a [slot][pixel] table;
//   * GAUSSIAN phase (lane = Gaussian slot x half of the region), run when 16 slots are full: every lane walks 16
//     pixels of ITS Gaussian, re-forms the WHITENED offsets (u, v) = L^T (pixel - mean) from the slot's record
//     (gs_raster.cuh: |u|, |v| <= ~4 wherever gp != 0) and accumulates the 10 sums (moments of gp in (u, v); w-weighted
//     upstream colour / depth gradients) in registers -- no cross-lane reduction except one SHFL per sum to join the
//     two halves -- and the 16 x 10 totals leave through shared memory as coalesced RED.ADD.F32.  Moments in the
//     whitened frame are well conditioned for any footprint: dL/dSigma' = L M2 L^T / (2 k^2) needs no cancellation
//     (moments of dx, dy lost 3 digits on 1000:1 footprints through -Q gQ Q).
#include "gs_internal.cuh"
#include "gs_raster.cuh"

namespace gs {

#ifndef GS_BWD_RING_STAGES
#define GS_BWD_RING_STAGES 2
#endif
#ifndef GS_BWD_RING_DELAY
#define GS_BWD_RING_DELAY 0
#endif
#ifndef GS_BWD_BATCH
#define GS_BWD_BATCH 128
#endif
constexpr int kTileBatch = GS_BWD_BATCH, kPadIdx = kTileBatch;  // list entries staged per round by a CTA; padding record
constexpr int kStages = GS_BWD_RING_STAGES, kDelay = GS_BWD_RING_DELAY, kAhead = kStages - kDelay;  // gs_raster.cuh
static_assert(kDelay >= 0 && kAhead >= 2, "ring shape");
#ifndef GS_BWD_MIN_CTAS
#define GS_BWD_MIN_CTAS 3
#endif
constexpr int kSlots = 16;     // Gaussians per flush of the Gaussian phase
constexpr int kPairRow = 33;   // float2 per slot row (32 pixels + 1: conflict-free transposed LDS.64)
constexpr int kOutVals = 10;   // sums per Gaussian (gs_internal.cuh kG2D, first 10)

// Record of the Gaussian in slot s, parked in shared memory by lane 0 of the pixel phase (one STS.128; up to round-2 v8
// the records were kept in registers of lane s through selects: 9 instructions per entry and 10 % of the stall samples,
// profiles/r2_v9_ring.md): the tile-local whitened offset of the instance and its list word (visible slot << 8 | mask).
// L is re-read from the feature record at the flush (one LDG.128 per lane per 16 Gaussians).
struct __align__(16) SlotRec { float u0, v0; uint32_t ent, pad; };

// Gaussian phase.  SPLIT = 2: lane = (slot = lane & 15, half = lane >> 4), 2 pixel rows per lane;
//                  SPLIT = 4: lane = (slot = lane & 7, quarter = lane >> 3), 1 pixel row per lane (tail flush, <= 8 slots).
// (xo, yo): tile-local coordinates of the region's first pixel.
// The moments of gp are accumulated in the REGION-CENTRED PIXEL coordinates (x, y) = (c - 3.5, row - 1.5): per pixel that
// is three operations with immediates (sum gp, sum gp x, sum gp x^2 per row; y enters once per row) instead of nine on
// per-Gaussian whitened offsets, and the six raw moments are mapped to the whitened frame once per Gaussian:
//   u = l11 x + l21 y + uc,  v = l22 y + vc     (uc, vc: whitened offset of the region's centre)
// |l| <= sqrt(0.5 log2(e) / 0.3) = 1.55 (the 0.3-pixel dilation bounds the conic) and |u|, |v| <= 2.9 wherever gp != 0, so
// |uc|, |vc| <= ~11 and the expansion of sum gp u^2 cancels at most ~1e2 x: 1e-5 relative, against the 1e-3 gradient bound.
template <int SPLIT>
__device__ __forceinline__ void gaussian_phase(float2* s_pair, const float4* s_pix, const SlotRec* s_slot, int nslot,
                                               int lane, float xo, float yo, const float4* __restrict__ feat,
                                               float* __restrict__ g2d) {
  constexpr int LS = 32 / SPLIT, R = 4 / SPLIT;  // slots per pass, pixel rows per lane
  __syncwarp();
  const int slot = lane & (LS - 1), part = lane / LS;
  const SlotRec sr = s_slot[slot];
  const uint32_t id = sr.ent >> 8;
  float4 L = make_float4(0.f, 0.f, 0.f, 0.f);
  if (slot < nslot) L = __ldg(feat + 3 * (size_t)id + 1);  // l11, l21, l22
  const float2* pr = s_pair + slot * kPairRow + part * (R * 8);
  const float4* px = s_pix + part * (R * 8);
  float m00 = 0.f, m10 = 0.f, m20 = 0.f, m01 = 0.f, m11 = 0.f, m02 = 0.f, c0 = 0.f, c1 = 0.f, c2 = 0.f, c3 = 0.f;
#pragma unroll
  for (int r = 0; r < R; ++r) {
    float s0 = 0.f, s1 = 0.f, s2 = 0.f;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      const float2 pw = pr[r * 8 + c];  // gp, w of (this Gaussian, pixel)
      const float4 gu = px[r * 8 + c];  // upstream dL/dRGB, dL/dDepth of the pixel
      constexpr float kHalf = 3.5f;
      const float x = (float)c - kHalf;
      s0 += pw.x;
      s1 = fmaf(pw.x, x, s1);
      s2 = fmaf(pw.x, x * x, s2);
      c0 = fmaf(pw.y, gu.x, c0);
      c1 = fmaf(pw.y, gu.y, c1);
      c2 = fmaf(pw.y, gu.z, c2);
      c3 = fmaf(pw.y, gu.w, c3);
    }
    const float y = (float)(part * R + r) - 1.5f;
    m00 += s0; m10 += s1; m20 += s2;
    m01 = fmaf(y, s0, m01); m11 = fmaf(y, s1, m11); m02 = fmaf(y * y, s0, m02);
  }
  float acc[kOutVals] = {m10, m01, m20, m11, m02, m00, c0, c1, c2, c3};
#pragma unroll
  for (int u = 0; u < kOutVals; ++u) {
    acc[u] += __shfl_xor_sync(kFull, acc[u], 16);
    if (SPLIT == 4) acc[u] += __shfl_xor_sync(kFull, acc[u], 8);
  }
  // raw moments -> whitened moments
  {
    const float M10 = acc[0], M01 = acc[1], M20 = acc[2], M11 = acc[3], M02 = acc[4], M00 = acc[5];
    const float xc = xo + 3.5f, yc = yo + 1.5f;
    const float uc = fmaf(L.x, xc, fmaf(L.y, yc, sr.u0)), vc = fmaf(L.z, yc, sr.v0);
    const float a1 = fmaf(L.x, M10, L.y * M01);                 // sum gp (l11 x + l21 y)
    const float b1 = L.z * M01;                                 // sum gp l22 y
    const float a2 = fmaf(L.x * L.x, M20, fmaf(2.f * L.x * L.y, M11, L.y * L.y * M02));
    const float ab = L.z * fmaf(L.x, M11, L.y * M02);
    const float b2 = L.z * L.z * M02;
    acc[0] = fmaf(uc, M00, a1);
    acc[1] = fmaf(vc, M00, b1);
    acc[2] = fmaf(uc, fmaf(uc, M00, 2.f * a1), a2);
    acc[3] = fmaf(vc, a1, fmaf(uc, fmaf(vc, M00, b1), ab));
    acc[4] = fmaf(vc, fmaf(vc, M00, 2.f * b1), b2);
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
    if (idx < total) atomicAdd(g2d + (size_t)(s_slot[sl_i].ent >> 8) * kG2D + val, s_out[idx]);
  }
  __syncwarp();
}

// NW: warps (= regions) per CTA, as in the forward (gs_raster.cu).
#ifndef GS_BWD_WARPS
#define GS_BWD_WARPS 4
#endif

template <int NW, bool HAS_GA>
__global__ void __launch_bounds__(NW * 32, (GS_BWD_MIN_CTAS * 8) / NW)
raster_bwd_kernel(int W, int H, int tiles_x, const uint32_t* __restrict__ order, const uint2* __restrict__ ranges,
                  const float4* __restrict__ inst, const float4* __restrict__ feat,
                  float bg0, float bg1, float bg2, const float* __restrict__ final_T,
                  const uint32_t* __restrict__ n_contrib, const float* __restrict__ d_rgb,
                  const float* __restrict__ d_depth, const float* __restrict__ d_alpha, float* __restrict__ g2d) {
  constexpr int CPT = 8 / NW;  // CTAs per tile
  constexpr int TPE = Ring<NW, kStages, kTileBatch>::TPE;
  __shared__ __align__(16) Ring<NW, kStages, kTileBatch> ring;  // staging ring (gs_raster.cuh): no block-wide barrier in the loop
  // per warp: byte offsets (into the stage) of the round's relevant entries, back to front
  __shared__ __align__(8) uint16_t s_idx[NW][kTileBatch + kGroup];
  __shared__ __align__(16) float2 s_pair_all[NW][kSlots * kPairRow];
  __shared__ __align__(16) float4 s_pix_all[NW][32];
  __shared__ SlotRec s_slot_all[NW][kSlots];
  __shared__ int s_nmax[NW];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  pdl_enter();
  const int tile = (int)__ldg(order + blockIdx.x / CPT), sub = (blockIdx.x % CPT) * NW + warp;
  const int tx0 = (tile % tiles_x) * GS_TILE, ty0 = (tile / tiles_x) * GS_TILE;
  const int xo = (sub % 2) * 8, yo = (sub / 2) * 4;
  const int X = xo + (lane & 7), Y = yo + (lane >> 3);  // tile-local pixel of this lane
  const float fx0 = (float)X, fy0 = (float)Y;
  const uint2 range = ranges[tile];
  const size_t HW = (size_t)W * H;
  float2* s_pair = s_pair_all[warp];
  float4* s_pix = s_pix_all[warp];
  SlotRec* s_slot = s_slot_all[warp];
  float T = 1.f, gC0 = 0.f, gC1 = 0.f, gC2 = 0.f, gD = 0.f, gA = 0.f;
  uint32_t last = 0;
  if (tx0 + X < W && ty0 + Y < H) {
    const size_t p = (size_t)(ty0 + Y) * W + (tx0 + X);
    T = final_T[p];
    last = n_contrib[p];
    gC0 = d_rgb[p]; gC1 = d_rgb[HW + p]; gC2 = d_rgb[2 * HW + p];
    if (d_depth) gD = d_depth[p];
    if (HAS_GA) gA = d_alpha[p];
  }
  s_pix[lane] = make_float4(gC0, gC1, gC2, gD);
  float S = T * (gC0 * bg0 + gC1 * bg1 + gC2 * bg2);
  const int n_w = (int)__reduce_max_sync(kFull, last);  // deepest blended list position of the region
  if (lane == 0) s_nmax[warp] = n_w;
  ring.init(tid);
  __syncthreads();
  int n = 0;
#pragma unroll
  for (int k = 0; k < NW; ++k) n = max(n, s_nmax[k]);  // ... and of the CTA: entries beyond it are never staged
  const int nb = (n + kTileBatch - 1) / kTileBatch;
  int nslot = 0;
  float2* pair_ptr = s_pair + lane;     // where this lane's (gp, w) of the next slot goes

  // producer state: rounds are staged back to front (staged round k = list round nb - 1 - k); this thread stages entry
  // e_pro of every round and fetches its list word one step ahead
  const int e_pro = tid / TPE;
  uint32_t v_pre = 0;
  auto fetch = [&](int k) {
    const int i = (nb - 1 - k) * kTileBatch + e_pro;
    v_pre = (i >= 0 && i < n) ? __float_as_uint(__ldg(&inst[range.x + i].z)) : 0u;
  };
  fetch(0);
#pragma unroll
  for (int k = 0; k < kAhead; ++k) {
    if (k < nb) ring.produce(k, (nb - 1 - k) * kTileBatch + e_pro, n, range.x, v_pre, tid, inst, feat);
    fetch(k + 1);
  }
  for (int k = 0; k < nb; ++k) {  // list rounds, back to front
    const int stage = k & (kStages - 1);
    const int pbase = (nb - 1 - k) * kTileBatch;
    if (pbase < n_w) {  // else nothing of this round was blended in this region
      mbar_wait(&ring.full[stage], (uint32_t)(k / kStages) & 1u);
      const StageBuf<kTileBatch>& sb = ring.st[stage];
      // the entries of this round that can reach this warp's region and lie in front of its deepest blended position, as
      // a list of byte offsets in REVERSE list order
      constexpr int NCH = kTileBatch / 32;
      bool rr[NCH];
      unsigned bb[NCH];
      int nrel = 0;
#pragma unroll
      for (int c = 0; c < NCH; ++c) {
        rr[c] = ((sb.rec[lane + 32 * c].ent >> sub) & 1u) && pbase + 32 * c + lane < n_w;
        bb[c] = __ballot_sync(kFull, rr[c]);
        nrel += __popc(bb[c]);
      }
      if (nrel) {
        const unsigned gt = ~((2u << lane) - 1u);  // lanes above this one
        uint16_t* idx = s_idx[warp];
        int at = 0;
#pragma unroll
        for (int c = NCH - 1; c >= 0; --c) {
          if (rr[c]) idx[at + __popc(bb[c] & gt)] = (uint16_t)((32 * c + lane) * 48);
          at += __popc(bb[c]);
        }
        if (lane < kGroup) idx[nrel + lane] = (uint16_t)(kPadIdx * 48);
        __syncwarp();
        const int lastb48 = ((int)last - pbase) * 48;  // entries of this round at offsets < lastb48 were blended by this pixel
        const char* recs = reinterpret_cast<const char*>(sb.rec);
        for (int r = 0; r < nrel; r += kGroup) {  // back to front, four list entries at a time
          const uint2 o4 = *reinterpret_cast<const uint2*>(idx + r);
          const uint32_t off[kGroup] = {o4.x & 0xffffu, o4.x >> 16, o4.y & 0xffffu, o4.y >> 16};
          float4 uv[kGroup];  // u0, v0, bits(list word), -
          float p[kGroup];
          bool hit[kGroup];
          unsigned bal[kGroup];
#pragma unroll
          for (int q = 0; q < kGroup; ++q) {
            const StageRec& e = *reinterpret_cast<const StageRec*>(recs + off[q]);
            const float4 a0 = e.g;  // l11, l21, l22, lo
            uv[q] = *reinterpret_cast<const float4*>(&e.uv);  // one LDS.128 brings the list word along
            p[q] = eval_power(uv[q].x, uv[q].y, a0.x, a0.y, a0.z, a0.w, fx0, fy0);
            // blended by the forward: alpha >= 1/255 and in front of the pixel's last contributor
            hit[q] = p[q] >= GS_POWER_MIN && (int)off[q] < lastb48;
            bal[q] = __ballot_sync(kFull, hit[q]);
          }
#pragma unroll
          for (int q = 0; q < kGroup; ++q) {
            if (bal[q] == 0) continue;  // the Gaussian reaches no pixel of the region
            const StageRec& e = *reinterpret_cast<const StageRec*>(recs + off[q]);
            // branch-free: a lane that is not hit runs the same instructions with alpha = 0 (T, S unchanged, gp = w = 0)
            const float4 f2 = e.c;
            const float og = ex2_approx(p[q]);  // opacity * G: log2(opacity) is folded into the exponent
            const float a = hit[q] ? fminf(GS_ALPHA_MAX, og) : 0.f;
            const float ioma = rcp_approx(1.f - a);
            T *= ioma;  // transmittance in front of this Gaussian
            const float w = a * T;
            float wi = fmaf(gC0, f2.x, fmaf(gC1, f2.y, fmaf(gC2, f2.z, gD * f2.w)));
            if (HAS_GA) wi += gA;
            const float dalpha = fmaf(T, wi, -S * ioma);
            S = fmaf(wi, w, S);
            const float gp = (og <= GS_ALPHA_MAX) ? a * dalpha : 0.f;  // no gradient through the clamp (Q2)
            *pair_ptr = make_float2(gp, w);
            pair_ptr += kPairRow;
            if (lane == 0) *reinterpret_cast<float4*>(s_slot + nslot) = uv[q];
            ++nslot;
          }
          // flush once per group of four entries, as soon as another group might not fit (one copy of the Gaussian phase
          // in the instruction stream instead of four)
          if (nslot > kSlots - kGroup) {
            gaussian_phase<2>(s_pair, s_pix, s_slot, nslot, lane, (float)xo, (float)yo, feat, g2d);
            nslot = 0;
            pair_ptr = s_pair + lane;
          }
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&ring.empty[stage]);  // this warp is done with the stage
    // refill: the stage of staged round k - kDelay takes round k + kAhead once every warp has released it
    const int kn = k + kAhead;
    if (kn < nb) {
      if (k >= kDelay) mbar_wait(&ring.empty[kn & (kStages - 1)], (uint32_t)((k - kDelay) / kStages) & 1u);
      ring.produce(kn, (nb - 1 - kn) * kTileBatch + e_pro, n, range.x, v_pre, tid, inst, feat);
      fetch(kn + 1);
    }
  }
  cp_async_wait_all();
  if (nslot > 8) gaussian_phase<2>(s_pair, s_pix, s_slot, nslot, lane, (float)xo, (float)yo, feat, g2d);
  else if (nslot > 0) gaussian_phase<4>(s_pair, s_pix, s_slot, nslot, lane, (float)xo, (float)yo, feat, g2d);
}

int launch_raster_bwd(gs_ctx* ctx, cudaStream_t s, const float* d_rgb, const float* d_depth, const float* d_alpha) {
  const int tiles = ctx->cam.tiles_x * ctx->cam.tiles_y;
  if (tiles == 0) return GS_OK;
  constexpr int NW = GS_BWD_WARPS;
#define GS_BWD(GA)                                                                                                  \
  GS_LAUNCH_PDL((raster_bwd_kernel<NW, GA>), tiles * (8 / NW), NW * 32, 0, s, ctx->cam.W, ctx->cam.H, ctx->cam.tiles_x, \
                (const uint32_t*)ctx->tile_order, (const uint2*)ctx->ranges, (const float4*)ctx->inst_rec, (const float4*)ctx->feat,    \
                ctx->bg[0], ctx->bg[1], ctx->bg[2],                                                                       \
                (const float*)ctx->final_T, (const uint32_t*)ctx->n_contrib, d_rgb, d_depth, d_alpha, ctx->g2d)
  if (d_alpha) GS_BWD(true); else GS_BWD(false);
#undef GS_BWD
  GS_LAUNCH_CHECK("raster_bwd_kernel");
  return GS_OK;
}

}  // namespace gs

// gs_raster.cuh -- pieces shared by the binning masks and the forward / backward compositing kernels.
//
// The power of a Gaussian at a pixel is evaluated in WHITENED, TILE-LOCAL form ("precision"):
//     p2 = lo - u^2 - v^2,   u = l11 X + l21 Y + u0,   v = l22 Y + v0,      alpha = min(0.99, 2^p2)
// with (X, Y) the pixel's coordinates inside its 16x16 tile (0..15), L = sqrt(0.5 log2 e) chol(conic) from gs_preprocess
// (fp64 there), lo = log2(opacity), and (u0, v0) = -L^T (mean - tile origin) formed in fp64 once per tile instance by
// gs_bin_tiles.  Every fp32 operand of the per-pixel arithmetic is then O(10) whatever the footprint's size or
// anisotropy (the direct form A dx^2 + B dx dy + C dy^2 cancels terms of size |A| dx^2 -- measured 1e-3 image error on
// config 5).  alpha >= 1/255 <=> p2 >= -log2(255): a constant, so neither the opacity nor a per-Gaussian threshold is
// read in the pixel loop.  The sequence below MUST be the same instructions in the forward and in the backward (the
// backward re-takes the forward's decisions), hence the explicit rounding intrinsics.
#pragma once

#include "gs_internal.cuh"

namespace gs {

constexpr unsigned kFull = 0xffffffffu;
constexpr int kGroup = 4;        // relevant entries evaluated together in the pixel loop
// Staging ring shape: STAGES stages (a power of two) of BATCH list entries.  A warp that has finished round j refills the
// stage of round j - DELAY (with round j - DELAY + STAGES): the warps of a CTA may be up to DELAY + 1 rounds apart before
// one waits for another, and STAGES - DELAY rounds are in flight.  The two compositing kernels choose differently (each
// defines kTileBatch / kStages / kDelay / kAhead in its own translation unit).  The forward is short of nothing but issue
// slots: rounds of 128 entries halve its per-round work (ballots, list building, barrier traffic, refill: 10 of its 34
// instructions per relevant entry), 4 stages / 2 rounds of slack (64 x 4 / 2 -> 64 x 8 / 5 -> 128 x 4 / 2: 61.9 -> 57.7 ->
// 55.0 us).  The backward pays for shared memory with a CTA of occupancy (64 x 8 / 2: 141.5 -> 154.3 us, 128 x 4 / 2: 115.1 ->
// 127.6 us) and spends its 12 KB on two stages of 128 entries, no slack (64 x 4 / 2 -> 128 x 2 / 0: 115.1 -> 112.3 us): the
// halved per-round work outweighs the tighter coupling of its four warps.
// One staged list entry (48 B): what the pixel loops read as broadcast LDS.128 x 2 + LDS.64.
//   g  = { l11, l21, l22, lo }, c = { r, g, b, z }   gathered by visible slot (cp.async.cg, 2 x 16 B)
//   { uv = { u0, v0 }, ent, pad }                     the 16-byte instance record written by the sort epilogue, one
//                                                     cp.async.cg: tile-local whitened offset + list word
//   ent = visible slot << 8 | region mask             (0 beyond the end of the list)
struct __align__(16) StageRec {
  float4 g, c;
  float2 uv;
  uint32_t ent, pad;
};
static_assert(sizeof(StageRec) == 48, "StageRec layout");
// One stage of a CTA's staging ring: kTileBatch consecutive list entries of the tile + the padding record
// (128 per round in both compositing kernels since v10; each kernel defines kTileBatch and kPadIdx).
template <int kTileBatch>
struct __align__(16) StageBuf {
  StageRec rec[kTileBatch + 1];  // [kTileBatch] = the padding record (never passes: lo = -inf)
};

// -log2(255): alpha >= 1/255  <=>  p2 >= kPowerMin
#define GS_POWER_MIN (-7.994353436858858f)

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  // .cg: the 16-byte gathers go straight from L2 to shared memory without allocating in L1 (the l1tex pipe is the
  // second limit of the compositing kernels: .ca -> .cg raster_fwd 63.2 -> 61.5 us, raster_bwd 119.6 -> 118.0 us)
#ifdef GS_CP_CA
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
#else
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
#endif
}
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gmem_src) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gmem_src) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
// TMA (bulk-copy engine) variant of the record gather, -DGS_RING_BULK: one cp.async.bulk of the 32 contiguous bytes
// {l11,l21,l22,lo}{r,g,b,z} per staged entry, completing on the stage's mbarrier through its transaction count, instead of
// two 16-byte cp.async.  Measured against the default in profiles/r2_v10_chain.md ("TMA where it pays").
__device__ __forceinline__ void bulk_copy32(void* smem_dst, const void* gmem_src, uint64_t* bar) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst), b = (uint32_t)__cvta_generic_to_shared(bar);
  asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], 32;" ::"r"(b) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], 32, [%2];" ::"r"(d), "l"(gmem_src), "r"(b) : "memory");
}

// mbarrier (shared::cta) helpers of the staging ring.  full[s]: every thread of the CTA arrives through
// cp.async.mbarrier.arrive.noinc, i.e. when ITS cp.async copies into stage s have landed (count = threads of the CTA);
// empty[s]: one arrival per warp that has finished reading stage s (count = warps of the CTA).
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared::cta.b64 st, [%0];\n}" ::"r"((uint32_t)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void cp_async_mbar_arrive(uint64_t* bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"((uint32_t)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
               : "=r"(ok) : "r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {}
}

// The staging ring shared by the forward and the backward kernels.  Every thread of the CTA is a producer: the entries
// of a round are dealt to the threads of the CTA (record halves g, c and the 16-byte instance record {u0, v0, list word}
// by one 16-byte cp.async.cg each), and every thread then lets full[stage] count its copies
// (cp.async.mbarrier.arrive.noinc).  Consumers (the same warps) wait on full[stage] and release the stage through
// empty[stage]; there is NO block-wide barrier in the loop: warps of different regions, which find different numbers of
// relevant entries per round, drift up to kDelay + 1 rounds apart (the per-round __syncthreads of v7 held 19-25 % of the
// stall samples of both kernels).
template <int NW, int kStages, int kTileBatch>
struct Ring {
  static constexpr int kPadIdx = kTileBatch;
  static_assert((kStages & (kStages - 1)) == 0, "ring depth must be a power of two");
  static constexpr int T = NW * 32, TPE = T / kTileBatch;  // threads per staged entry: 1, 2 or 4
  static_assert(TPE == 1 || TPE == 2 || TPE == 4, "2, 4 or 8 warps");
  StageBuf<kTileBatch> st[kStages];
  uint64_t full[kStages], empty[kStages];

  __device__ __forceinline__ void init(int tid) {
    if (tid < kStages) {  // padding records never pass: lo = -inf  =>  p2 = -inf
      StageRec& pr = st[tid].rec[kPadIdx];
      pr.g = make_float4(0.f, 0.f, 0.f, -INFINITY);
      pr.c = make_float4(0.f, 0.f, 0.f, 0.f);
      pr.uv = make_float2(0.f, 0.f);
      pr.ent = 0u;
      mbar_init(&full[tid], T);
      mbar_init(&empty[tid], NW);
    }
  }
  // stages list entry i (valid if i < n) of the tile whose list starts at `first`, for staged round k; v = ids[first + i]
  __device__ __forceinline__ void produce(int k, int i, int n, uint32_t first, uint32_t v, int tid,
                                          const float4* __restrict__ inst, const float4* __restrict__ feat) {
    const int stage = k & (kStages - 1), part = tid & (TPE - 1);
    StageRec& r = st[stage].rec[tid / TPE];
    if (i >= 0 && i < n) {
      const float4* src = feat + 3 * (size_t)(v >> 8) + 1;
#ifdef GS_RING_BULK
      if (part == 0) bulk_copy32(&r.g, src, &full[stage]);
#else
      if (part == 0) cp_async16(&r.g, src);
      if (part == (1 & (TPE - 1))) cp_async16(&r.c, src + 1);
#endif
      if (part == (2 & (TPE - 1))) cp_async16(&r.uv, inst + first + i);  // {u0, v0, list word, -}: the record's last 16 bytes
    }
    cp_async_mbar_arrive(&full[stage]);
  }
};

// Feature record -> whitened offset relative to the origin (ox, oy), in fp64 (exact integer part of the mean, exact
// products with the fp32-rounded L; one rounding of u0, v0 at the end).  Also returns the origin-relative mean (fp32).
__device__ __forceinline__ void decode_whitened(const float4& f0, const float4& f1, int ox, int oy, float& u0, float& v0,
                                                float& mx, float& my) {
  const int pk = __float_as_int(f0.z);
  const double mxd = (double)(((pk << 16) >> 16) - ox) + (double)f0.x;
  const double myd = (double)((pk >> 16) - oy) + (double)f0.y;
  u0 = (float)(-((double)f1.x * mxd + (double)f1.y * myd));
  v0 = (float)(-((double)f1.z * myd));
  mx = (float)mxd;
  my = (float)myd;
}

// p2 at the lane's pixel (fx0, fy0) of the tile: five FFMA, no subtraction of large numbers
__device__ __forceinline__ float eval_power(float u0, float v0, float l11, float l21, float l22, float lo, float fx0,
                                            float fy0) {
  const float u = __fmaf_rn(l11, fx0, __fmaf_rn(l21, fy0, u0));
  const float v = __fmaf_rn(l22, fy0, v0);
  return __fmaf_rn(-u, u, __fmaf_rn(-v, v, lo));
}

// Which of the eight 8x4-pixel regions of a 16x16 tile can the ellipse {p2 >= -log2(255)} reach?  Exact up to an
// outward slack: per band of four pixel rows the ellipse's x-extent over the band is [xl, xr] (a convex set projects
// to an interval, attained at the band-clamped extreme points), and a region is hit iff the interval meets the
// region's columns.  (mx, my): mean relative to the tile origin.  Square roots and reciprocals are the 1-instruction
// approximations (2 ulp): the test has 0.02 of slack in the exponent.  ~70 instructions per (Gaussian, tile) instance after a
// per-Gaussian setup; the previous per-rectangle maximisation of the quadratic was ~500 and made the duplication kernel
// issue-bound.
__device__ __forceinline__ float sqrt_approx(float x) {
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// Per-Gaussian part of the region test (the same for every tile of the Gaussian's rectangle).
struct MaskSetup { float R2, hy, dyR, il11, l21, l22; };
__device__ __forceinline__ MaskSetup region_mask_setup(float l11, float l21, float l22, float lo) {
  MaskSetup m;
  m.R2 = lo - GS_POWER_MIN + 0.02f;   // outward slack: 0.02 in the exponent, >> the error of the approximate ops below
  const float R = sqrt_approx(fmaxf(m.R2, 0.f)), il22 = rcp_approx(l22);
  m.hy = R * il22;                                                    // half height of the ellipse
  m.dyR = -l21 * R * rsqrtf(l21 * l21 + l22 * l22) * il22;            // row (relative to the mean) of the rightmost point
  m.il11 = rcp_approx(l11); m.l21 = l21; m.l22 = l22;
  return m;
}

__device__ __forceinline__ uint32_t region_mask(const MaskSetup& g, float mx, float my) {
  if (!(g.R2 > 0.f)) return 0u;
  const float eps = 2e-3f + 2e-6f * fabsf(mx);
  uint32_t m = 0;
#pragma unroll
  for (int band = 0; band < 4; ++band) {
    const float ya = (float)(4 * band) - my, yb = ya + 3.f;
    const float lo_y = fmaxf(ya, -g.hy), hi_y = fminf(yb, g.hy);
    if (lo_y > hi_y) continue;
    const float dyr = fminf(fmaxf(g.dyR, lo_y), hi_y), dyl = fminf(fmaxf(-g.dyR, lo_y), hi_y);
    const float vr = g.l22 * dyr, vl = g.l22 * dyl;
    const float sr = sqrt_approx(fmaxf(g.R2 - vr * vr, 0.f)), sl = sqrt_approx(fmaxf(g.R2 - vl * vl, 0.f));
    const float xr = mx + (sr - g.l21 * dyr) * g.il11 + eps, xl = mx - (sl + g.l21 * dyl) * g.il11 - eps;
    if (xl <= 7.f && xr >= 0.f) m |= 1u << (2 * band);
    if (xl <= 15.f && xr >= 8.f) m |= 2u << (2 * band);
  }
  return m;
}

}  // namespace gs

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
constexpr int kTileBatch = 64;   // list entries staged per round by a CTA
constexpr int kStages = 3;       // staging ring depth
constexpr int kPadIdx = kTileBatch;  // index of the stage's padding record (never passes: lo = -inf)

// One staged list entry (48 B): what the pixel loops read as broadcast LDS.128 x 2 + LDS.64.
//   g  = { l11, l21, l22, lo }, c = { r, g, b, z }   gathered by visible slot (cp.async, 2 x 16 B)
//   uv = { u0, v0 }                                   the instance's tile-local whitened offset (cp.async 8 B)
//   ent = visible slot << 8 | region mask             (0 beyond the end of the list)
struct __align__(16) StageRec {
  float4 g, c;
  float2 uv;
  uint32_t ent, pad;
};
static_assert(sizeof(StageRec) == 48, "StageRec layout");
// One stage of a CTA's staging ring: 64 consecutive list entries of the tile + the padding record.
struct __align__(16) StageBuf {
  StageRec rec[kTileBatch + 1];
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
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gmem_src) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

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

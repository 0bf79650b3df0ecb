// gs_raster.cuh -- pieces shared by the forward and backward compositing kernels.  The alpha evaluation MUST be the
// same instruction sequence in both (the backward re-takes the forward's alpha >= 1/255 decisions), so it is written
// with explicit rounding intrinsics that the compiler cannot re-associate or contract differently per kernel.
#pragma once

#include "gs_internal.cuh"

namespace gs {

constexpr int kBatch = 256;  // Gaussians staged in shared memory per round (= threads per tile CTA)

// Staged Gaussian, tile-local: 3 x float4 (broadcast LDS.128 in the inner loop)
//   g0 = { mx_local, my_local, A, B }   g1 = { C, opacity, r, g }   g2 = { b, z, id (bits), - }
struct Staged {
  float4 g0, g1, g2;
};

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// power2 = A dx^2 + B dx dy + C dy^2 (log2 units, <= 0 up to rounding); returns opacity * 2^power2 (unclamped).
__device__ __forceinline__ float eval_og(float dx, float dy, float A, float B, float C, float o) {
  const float t = __fmaf_rn(A, dx, __fmul_rn(B, dy));
  float p = __fmul_rn(t, dx);
  p = __fmaf_rn(__fmul_rn(C, dy), dy, p);
  return __fmul_rn(o, ex2_approx(p));
}

// Gathers Gaussian `id` and converts its mean to coordinates local to the tile origin (ox, oy): the integer part of the
// mean minus the origin is exact, the fraction is added in fp32 (absolute pixel coordinates
// in fp32 would cost ~6e-5 px at x ~ 1000).
__device__ __forceinline__ void stage_gaussian(const float4* __restrict__ feat, uint32_t id, int ox, int oy,
                                               Staged& s) {
  const float4 f0 = __ldg(feat + 3 * (size_t)id);
  const float4 f1 = __ldg(feat + 3 * (size_t)id + 1);
  const float4 f2 = __ldg(feat + 3 * (size_t)id + 2);
  const float mx = (float)(__float_as_int(f0.z) - ox) + f0.x;
  const float my = (float)(__float_as_int(f0.w) - oy) + f0.y;
  s.g0 = make_float4(mx, my, f1.x, f1.y);
  s.g1 = make_float4(f1.z, f1.w, f2.x, f2.y);
  s.g2 = make_float4(f2.z, f2.w, __uint_as_float(id), 0.f);
}

// Thread -> pixel mapping inside a 16x16 tile: a warp covers an 8x4 patch (less early-exit waste than 16x2).
__device__ __forceinline__ void thread_pixel(int tid, int& lx, int& ly) {
  const int warp = tid >> 5, lane = tid & 31;
  lx = (warp & 1) * 8 + (lane & 7);
  ly = (warp >> 1) * 4 + (lane >> 3);
}

}  // namespace gs

// gs_raster.cuh -- pieces shared by the forward and backward compositing kernels (v2: one warp per tile region,
// several interleaved pixels per lane).  The power evaluation MUST be the same instruction sequence in both kernels
// (the backward re-takes the forward's alpha >= 1/255 decisions), so it is written with explicit rounding intrinsics
// that the compiler cannot contract or re-associate differently per kernel.
#pragma once

#include "gs_internal.cuh"

namespace gs {

constexpr int kWarpBatch = 32;  // Gaussians staged per round by one warp (one per lane)

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// Pixel slots of a lane.  Lanes form an 8 (x) by 4 (y) grid; slot (kx, ky) of lane (lx, ly) is the pixel
// (lx + 8 kx, ly + 4 ky) of the warp's region, kx < NX, ky < NY: the region is (8 NX) x (4 NY) pixels and a lane's
// pixels are INTERLEAVED over it, so that the footprint of one Gaussian falls on few slots of many lanes (SIMT
// efficiency) rather than on all slots of few lanes.  Slot index k = ky * NX + kx.

// One staged Gaussian, decoded for a region with origin (ox, oy).
struct GaussReg {
  float mx, my;       // mean, region-local
  float A, B, C, o;   // pre-scaled conic, opacity
  float thr;          // power threshold: alpha >= 1/255 <=> power2 >= thr
};

__device__ __forceinline__ void decode_gauss(const float4& f0, const float4& f1, int ox, int oy, GaussReg& g) {
  const int pk = __float_as_int(f0.z);
  g.mx = (float)(((pk << 16) >> 16) - ox) + f0.x;  // integer part minus origin is exact; fraction added in fp32
  g.my = (float)((pk >> 16) - oy) + f0.y;
  g.A = f1.x; g.B = f1.y; g.C = f1.z; g.o = f1.w;
  g.thr = f0.w;
}

// power2 of every slot: p[ky*NX+kx] = dx (A dx + B dy) + C dy^2, with the products shared across rows / columns.
// Explicit rounding intrinsics: the sequence is the same in every kernel that includes this header.
template <int NX, int NY>
__device__ __forceinline__ void eval_power(const GaussReg& g, float fx0, float fy0, float (&dx)[NX], float (&dy)[NY],
                                           float (&p)[NX * NY]) {
  float ax[NX], cy[NY];
#pragma unroll
  for (int kx = 0; kx < NX; ++kx) {
    dx[kx] = __fsub_rn(fx0 + 8.f * kx, g.mx);
    ax[kx] = __fmul_rn(g.A, dx[kx]);
  }
#pragma unroll
  for (int ky = 0; ky < NY; ++ky) {
    dy[ky] = __fsub_rn(fy0 + 4.f * ky, g.my);
    cy[ky] = __fmul_rn(__fmul_rn(g.C, dy[ky]), dy[ky]);
  }
#pragma unroll
  for (int ky = 0; ky < NY; ++ky)
#pragma unroll
    for (int kx = 0; kx < NX; ++kx)
      p[ky * NX + kx] = __fmaf_rn(dx[kx], __fmaf_rn(g.B, dy[ky], ax[kx]), cy[ky]);
}

// the same sequence for one pixel per lane (8x4 regions)
__device__ __forceinline__ float eval_power1(float mx, float my, float A, float B, float C, float fx0, float fy0,
                                             float& dx, float& dy) {
  dx = __fsub_rn(fx0, mx);
  dy = __fsub_rn(fy0, my);
  return __fmaf_rn(dx, __fmaf_rn(B, dy, __fmul_rn(A, dx)), __fmul_rn(__fmul_rn(C, dy), dy));
}

__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

constexpr unsigned kFull = 0xffffffffu;
constexpr int kGroup = 4;                    // Gaussians evaluated together in phase 2

// Maximum of power2 over the continuous rectangle [0,xmax] x [0,ymax] (region-local), exact for the concave quadratic:
// 0 if the centre is inside, else the largest of the four clamped edge maxima.
__device__ __forceinline__ float region_max_power(const GaussReg& g, float xmax, float ymax) {
  const float x0 = -g.mx, x1 = xmax - g.mx, y0 = -g.my, y1 = ymax - g.my;  // rectangle in centre-relative coordinates
  if (x0 <= 0.f && x1 >= 0.f && y0 <= 0.f && y1 >= 0.f) return 0.f;
  const float i2C = rcp_approx(2.f * g.C), i2A = rcp_approx(2.f * g.A);  // the test has 1e-3 of slack
  float best = -INFINITY;
#pragma unroll
  for (int e = 0; e < 2; ++e) {
    const float dxe = e ? x1 : x0;
    const float dys = fminf(fmaxf(-g.B * dxe * i2C, y0), y1);
    best = fmaxf(best, g.A * dxe * dxe + g.B * dxe * dys + g.C * dys * dys);
    const float dye = e ? y1 : y0;
    const float dxs = fminf(fmaxf(-g.B * dye * i2A, x0), x1);
    best = fmaxf(best, g.A * dxs * dxs + g.B * dxs * dye + g.C * dye * dye);
  }
  return best;
}

}  // namespace gs

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

// power2 of every slot: p[ky*NX+kx] = A dx^2 + B dx dy + C dy^2 with the products shared across rows / columns.
template <int NX, int NY>
__device__ __forceinline__ void eval_power(const GaussReg& g, float fx0, float fy0, float (&dx)[NX], float (&dy)[NY],
                                           float (&p)[NX * NY]) {
  float ax[NX], bx[NX], cy[NY];
#pragma unroll
  for (int kx = 0; kx < NX; ++kx) {
    dx[kx] = __fsub_rn(fx0 + 8.f * kx, g.mx);
    ax[kx] = __fmul_rn(__fmul_rn(g.A, dx[kx]), dx[kx]);
    bx[kx] = __fmul_rn(g.B, dx[kx]);
  }
#pragma unroll
  for (int ky = 0; ky < NY; ++ky) {
    dy[ky] = __fsub_rn(fy0 + 4.f * ky, g.my);
    cy[ky] = __fmul_rn(__fmul_rn(g.C, dy[ky]), dy[ky]);
  }
#pragma unroll
  for (int ky = 0; ky < NY; ++ky)
#pragma unroll
    for (int kx = 0; kx < NX; ++kx) p[ky * NX + kx] = __fmaf_rn(bx[kx], dy[ky], __fadd_rn(ax[kx], cy[ky]));
}

}  // namespace gs

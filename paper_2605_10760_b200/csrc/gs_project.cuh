// gs_project.cuh -- the per-Gaussian EWA projection chain in fp64 (used by gs_preprocess and recomputed by the
// per-Gaussian backward).  fp64 here is deliberate: the 2-D mean must be good to ~5e-8 px and
// the conic must not lose digits to cancellation for the 1e-5 absolute image tolerance; it costs ~250 DP flops per
// visible Gaussian in HBM-bound kernels.
#pragma once

#include "gs_internal.cuh"

namespace gs {

// R = double in gs_preprocess (the 2-D mean and the conic feed the 1e-5 image tolerance), float in the per-Gaussian
// backward (1e-3 gradient tolerance; fp32 halves the registers and the latency of the chain).
template <typename R>
struct Proj {
  R x, y, z;        // camera-space centre
  R r[4], qn;       // unit quaternion, |q|
  R Rm[9], M3[9];   // R(r), M3 = R diag(s)
  R J00, J02, J11, J12;
  R Tm[6], M[6];    // T = J W, M = T M3
  R cxx, cxy, cyy;  // Sigma' (dilated)
  R a, b, c;        // conic
  R mx, my;
};
using ProjD = Proj<double>;

// Canonical fp32 depth key: bit pattern of fmaf(W20, mx, fmaf(W21, my, fmaf(W22, mz, tz)))  (Q13).
__device__ __forceinline__ float depth_key_f32(const float* T, float mx, float my, float mz) {
  return __fmaf_rn(T[8], mx, __fmaf_rn(T[9], my, __fmaf_rn(T[10], mz, T[11])));
}

template <typename R>
__device__ __forceinline__ void quat_rotation(const R* r, R* Rm) {
  const R w = r[0], x = r[1], y = r[2], z = r[3];
  const R one = (R)1, two = (R)2;
  Rm[0] = one - two * (y * y + z * z); Rm[1] = two * (x * y - w * z);       Rm[2] = two * (x * z + w * y);
  Rm[3] = two * (x * y + w * z);       Rm[4] = one - two * (x * x + z * z); Rm[5] = two * (y * z - w * x);
  Rm[6] = two * (x * z - w * y);       Rm[7] = two * (y * z + w * x);       Rm[8] = one - two * (x * x + y * y);
}

// Returns false when the Gaussian is culled before any covariance work (behind the near plane, opacity < 1/255) or
// its projection is degenerate / non-finite.  CULL = false (per-Gaussian backward): visibility was already decided by
// gs_preprocess in fp64, so none of the early-outs is taken and every field of P is always written -- an fp32
// re-projection must never disagree with the forward about which Gaussians exist.
template <typename R, bool CULL = true>
__device__ __forceinline__ bool project_gaussian(const DevCam& cam, const float* T, float mu0, float mu1, float mu2,
                                                 float s0, float s1, float s2, float q0, float q1, float q2, float q3,
                                                 float opacity, Proj<R>& P) {
  const R W[9] = {(R)T[0], (R)T[1], (R)T[2], (R)T[4], (R)T[5], (R)T[6], (R)T[8], (R)T[9], (R)T[10]};
  const R m0 = mu0, m1 = mu1, m2 = mu2;
  P.x = W[0] * m0 + W[1] * m1 + W[2] * m2 + (R)T[3];
  P.y = W[3] * m0 + W[4] * m1 + W[5] * m2 + (R)T[7];
  P.z = W[6] * m0 + W[7] * m1 + W[8] * m2 + (R)T[11];
  if (CULL && !(P.z > (R)cam.near_z)) return false;
  if (CULL && (double)opacity < 1.0 / 255.0) return false;
  const R q[4] = {(R)q0, (R)q1, (R)q2, (R)q3};
  P.qn = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
  const R iq = (R)1 / P.qn;
#pragma unroll
  for (int k = 0; k < 4; ++k) P.r[k] = q[k] * iq;
  quat_rotation<R>(P.r, P.Rm);
  const R s[3] = {(R)s0, (R)s1, (R)s2};
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) P.M3[3 * r + c] = P.Rm[3 * r + c] * s[c];
  const R iz = (R)1 / P.z, fx = cam.fx, fy = cam.fy;
  P.J00 = fx * iz; P.J02 = -fx * P.x * iz * iz;
  P.J11 = fy * iz; P.J12 = -fy * P.y * iz * iz;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    P.Tm[c] = P.J00 * W[c] + P.J02 * W[6 + c];
    P.Tm[3 + c] = P.J11 * W[3 + c] + P.J12 * W[6 + c];
  }
#pragma unroll
  for (int r = 0; r < 2; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c)
      P.M[3 * r + c] = P.Tm[3 * r] * P.M3[c] + P.Tm[3 * r + 1] * P.M3[3 + c] + P.Tm[3 * r + 2] * P.M3[6 + c];
  P.cxx = P.M[0] * P.M[0] + P.M[1] * P.M[1] + P.M[2] * P.M[2] + (R)GS_DILATION;
  P.cxy = P.M[0] * P.M[3] + P.M[1] * P.M[4] + P.M[2] * P.M[5];
  P.cyy = P.M[3] * P.M[3] + P.M[4] * P.M[4] + P.M[5] * P.M[5] + (R)GS_DILATION;
  const R det = P.cxx * P.cyy - P.cxy * P.cxy;
  if (CULL && (!(det > (R)0) || !isfinite(det))) return false;
  const R idet = (R)1 / det;
  P.a = P.cyy * idet; P.b = -P.cxy * idet; P.c = P.cxx * idet;
  P.mx = fx * P.x * iz + (R)cam.cx;
  P.my = fy * P.y * iz + (R)cam.cy;
  if (CULL && (!isfinite(P.mx) || !isfinite(P.my))) return false;
  return true;
}

// Screen extent {alpha >= 1/255}: exact half widths rho sqrt(Sigma'_xx), rho sqrt(Sigma'_yy), rho^2 = 2 ln(255 o),
// padded outward by 2^-10 relative + 2^-7 px so that the fp32 rasteriser never sees alpha >= 1/255 outside the rect
// (the rendered result is then independent of binning; Q5).  Returns false if no pixel is covered.
__device__ __forceinline__ bool tile_rect(const DevCam& cam, const ProjD& P, float opacity, int& tx0, int& ty0,
                                          int& tx1, int& ty1) {
  // fp32 is enough here: its rounding (1e-7 relative, < 1e-4 px) is far inside the outward padding, and the fp64 log and
  // square roots were a third of the instructions of a visible thread
  const float rho = sqrtf(2.f * logf(255.f * opacity));
  const float hx = rho * sqrtf((float)P.cxx) * (1.f + 0.0009765625f) + 0.0078125f;
  const float hy = rho * sqrtf((float)P.cyy) * (1.f + 0.0009765625f) + 0.0078125f;
  const float mx = (float)P.mx, my = (float)P.my;
  const float Wd = (float)cam.W, Hd = (float)cam.H;
  const float x0 = fmaxf(0.f, ceilf(mx - hx)), x1 = fminf(Wd, floorf(mx + hx) + 1.f);
  const float y0 = fmaxf(0.f, ceilf(my - hy)), y1 = fminf(Hd, floorf(my + hy) + 1.f);
  if (!(x1 > x0) || !(y1 > y0)) return false;
  const int ix0 = (int)x0, ix1 = (int)x1, iy0 = (int)y0, iy1 = (int)y1;
  tx0 = ix0 / GS_TILE; ty0 = iy0 / GS_TILE;
  tx1 = (ix1 - 1) / GS_TILE + 1; ty1 = (iy1 - 1) / GS_TILE + 1;
  return true;
}

}  // namespace gs

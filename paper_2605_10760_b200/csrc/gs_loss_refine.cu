// gs_loss_refine.cu -- the refinement loss of the fused map, Eq. 23, on the exposure-compensated render
//     I~(u) = e^{a_k} I^(u) + b_k :    alpha' L1(I~, I) + lambda (1 - SSIM(I~, I)) + beta L1(D^, D-)
// fused so that a refinement iteration needs no framework ops between gs_rasterize_fwd and gs_rasterize_bwd: it writes the
// upstream gradients dL/dI^, dL/dD^ that gs_rasterize_bwd consumes, the gradients of the per-keyframe log-gain and bias
// (a_k, b_k), and the loss terms.  (The normal term lambda'_n L_normal is gs_loss_normal, gs_normals.cu.)
// Readings: Q19 SSIM = 11 x 11 Gaussian window, sigma 1.5, C1 = 0.01^2, C2 = 0.03^2, zero padding, per channel,
// mean over pixels and channels; Q18 mean reductions, depth term where the target depth is > 0, sign(0) = 0; Q16 the
// weights are call arguments (the paper's lambda_n is garbled).
// Two image passes (separable 11-tap window in shared memory, 16 x 16 pixel tiles with a 5-pixel halo):
//   pass 1: windowed moments of (I~, I) -> SSIM map (summed) and its partials w.r.t. the moments of I~  (9 H W floats of
//           caller-provided scratch);   pass 2: the window applied to the partials (the window is symmetric, zero padding
//           is self-adjoint) -> dSSIM/dI~, combined with the L1 term, times e^a -> dL/dI^; sums for dL/da, dL/db.
// HBM-bound: 36 floats per pixel in total.  Product code: nothing here includes, links or calls oracle/.
#include "gs_internal.cuh"

namespace gs {

constexpr int kWinR = 5, kWin = 11, kRT = 16, kRH = kRT + 2 * kWinR;  // window radius / size, tile, tile + halo
__constant__ float c_win[kWin];

__device__ __forceinline__ float sgnf(float d) { return d > 0.f ? 1.f : (d < 0.f ? -1.f : 0.f); }

template <int NV>
__device__ __forceinline__ void block_sum_atomic(double (&v)[NV], double* out) {
  __shared__ double s_v[8][NV];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < NV; ++k) {
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], d);
    if (lane == 0) s_v[warp][k] = v[k];
  }
  __syncthreads();
  if (threadIdx.x < NV) {
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < 8; ++w) t += s_v[w][threadIdx.x];
    if (t != 0.0) atomicAdd(out + threadIdx.x, t);
  }
}

// pass 1: one CTA = one 16x16 tile of one channel
__global__ void __launch_bounds__(256)
ssim_moments_kernel(int W, int H, const float* __restrict__ rgb, const float* __restrict__ trgb, const float* __restrict__ ab,
                    float* __restrict__ work, double* __restrict__ sums) {
  __shared__ float s_x[kRH][kRH + 1], s_y[kRH][kRH + 1];
  __shared__ float s_h[5][kRH][kRT + 1];
  const int c = blockIdx.z, tx0 = blockIdx.x * kRT, ty0 = blockIdx.y * kRT;
  const size_t HW = (size_t)W * H;
  const float ea = expf(__ldg(ab)), b = __ldg(ab + 1);
  const float* xs = rgb + c * HW;
  const float* ys = trgb + c * HW;
  for (int i = threadIdx.x; i < kRH * kRH; i += 256) {
    const int r = i / kRH, q = i - r * kRH, X = tx0 + q - kWinR, Y = ty0 + r - kWinR;
    const bool in = X >= 0 && X < W && Y >= 0 && Y < H;   // zero padding applies to the exposed image too
    s_x[r][q] = in ? fmaf(ea, xs[(size_t)Y * W + X], b) : 0.f;
    s_y[r][q] = in ? ys[(size_t)Y * W + X] : 0.f;
  }
  __syncthreads();
  for (int i = threadIdx.x; i < kRH * kRT; i += 256) {  // horizontal pass: 26 rows x 16 columns x 5 moments
    const int r = i / kRT, q = i - r * kRT;
    float m1 = 0.f, m2 = 0.f, e11 = 0.f, e22 = 0.f, e12 = 0.f;
#pragma unroll
    for (int k = 0; k < kWin; ++k) {
      const float w = c_win[k], x = s_x[r][q + k], y = s_y[r][q + k];
      m1 = fmaf(w, x, m1); m2 = fmaf(w, y, m2);
      e11 = fmaf(w * x, x, e11); e22 = fmaf(w * y, y, e22); e12 = fmaf(w * x, y, e12);
    }
    s_h[0][r][q] = m1; s_h[1][r][q] = m2; s_h[2][r][q] = e11; s_h[3][r][q] = e22; s_h[4][r][q] = e12;
  }
  __syncthreads();
  const int lx = threadIdx.x & 15, ly = threadIdx.x >> 4, X = tx0 + lx, Y = ty0 + ly;
  double ssum[1] = {0.0};
  if (X < W && Y < H) {
    float m[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int k = 0; k < kWin; ++k) {
      const float w = c_win[k];
#pragma unroll
      for (int u = 0; u < 5; ++u) m[u] = fmaf(w, s_h[u][ly + k][lx], m[u]);
    }
    const double m1 = m[0], m2 = m[1], e11 = m[2], e22 = m[3], e12 = m[4];
    const double C1 = 1e-4, C2 = 9e-4;
    const double n1 = 2 * m1 * m2 + C1, n2 = 2 * (e12 - m1 * m2) + C2;
    const double d1 = m1 * m1 + m2 * m2 + C1, d2 = (e11 - m1 * m1) + (e22 - m2 * m2) + C2;
    const double id = 1.0 / (d1 * d2), s = n1 * n2 * id;
    ssum[0] = s;
    const size_t p = (size_t)Y * W + X;
    work[(3 * c + 0) * HW + p] = (float)((2 * m2 * n2 - 2 * m2 * n1) * id - s * (2 * m1 / d1 - 2 * m1 / d2));  // ds/dm1
    work[(3 * c + 1) * HW + p] = (float)(-s / d2);                                                           // ds/de11
    work[(3 * c + 2) * HW + p] = (float)(2 * n1 * id);                                                        // ds/de12
  }
  block_sum_atomic<1>(ssum, sums + 1);
}

// pass 2: window applied to the partials, gradients and the remaining sums
__global__ void __launch_bounds__(256)
ssim_grad_kernel(int W, int H, const float* __restrict__ rgb, const float* __restrict__ depth, const float* __restrict__ trgb,
                 const float* __restrict__ tdepth, const float* __restrict__ ab, const float* __restrict__ work,
                 float w_l1, float w_ssim, float w_d, float* __restrict__ d_rgb, float* __restrict__ d_depth,
                 double* __restrict__ sums) {
  __shared__ float s_p[3][kRH][kRH + 1];
  __shared__ float s_h[3][kRH][kRT + 1];
  const int c = blockIdx.z, tx0 = blockIdx.x * kRT, ty0 = blockIdx.y * kRT;
  const size_t HW = (size_t)W * H;
  const float ea = expf(__ldg(ab)), b = __ldg(ab + 1);
  for (int i = threadIdx.x; i < kRH * kRH; i += 256) {
    const int r = i / kRH, q = i - r * kRH, X = tx0 + q - kWinR, Y = ty0 + r - kWinR;
    const bool in = X >= 0 && X < W && Y >= 0 && Y < H;
    const size_t p = (size_t)Y * W + X;
#pragma unroll
    for (int u = 0; u < 3; ++u) s_p[u][r][q] = in ? work[(3 * c + u) * HW + p] : 0.f;
  }
  __syncthreads();
  for (int i = threadIdx.x; i < kRH * kRT; i += 256) {
    const int r = i / kRT, q = i - r * kRT;
    float a0 = 0.f, a1 = 0.f, a2 = 0.f;
#pragma unroll
    for (int k = 0; k < kWin; ++k) {
      const float w = c_win[k];
      a0 = fmaf(w, s_p[0][r][q + k], a0); a1 = fmaf(w, s_p[1][r][q + k], a1); a2 = fmaf(w, s_p[2][r][q + k], a2);
    }
    s_h[0][r][q] = a0; s_h[1][r][q] = a1; s_h[2][r][q] = a2;
  }
  __syncthreads();
  const int lx = threadIdx.x & 15, ly = threadIdx.x >> 4, X = tx0 + lx, Y = ty0 + ly;
  double v[4] = {0.0, 0.0, 0.0, 0.0};  // sum |I~ - I|, sum dL/dI~ e^a I^, sum dL/dI~, sum |D^ - D|
  if (X < W && Y < H) {
    float a0 = 0.f, a1 = 0.f, a2 = 0.f;
#pragma unroll
    for (int k = 0; k < kWin; ++k) {
      const float w = c_win[k];
      a0 = fmaf(w, s_h[0][ly + k][lx], a0); a1 = fmaf(w, s_h[1][ly + k][lx], a1); a2 = fmaf(w, s_h[2][ly + k][lx], a2);
    }
    const size_t p = (size_t)Y * W + X;
    const float x = rgb[c * HW + p], y = trgb[c * HW + p];
    const float xt = fmaf(ea, x, b), d = xt - y;
    // dL/dI~ = alpha' sign(I~ - I) / (3 H W) - lambda dSSIM/dI~,  dSSIM/dI~ = (W*A + 2 I~ W*B + I W*C) / (3 H W)
    const float g = w_l1 * sgnf(d) - w_ssim * (a0 + 2.f * xt * a1 + y * a2);
    d_rgb[c * HW + p] = ea * g;
    v[0] = (double)fabsf(d); v[1] = (double)(g * ea * x); v[2] = (double)g;
    if (c == 0) {
      const float t = tdepth[p];
      const float dd = t > 0.f ? depth[p] - t : 0.f;
      d_depth[p] = w_d * sgnf(dd);
      v[3] = (double)fabsf(dd);
    }
  }
  block_sum_atomic<4>(v, sums + 2);
}

__global__ void refine_final_kernel(double* sums, double inv_n, double inv_p, double alpha_p, double lambda, double beta,
                                    float* g_ab) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  // raw: [1] sum SSIM map, [2] sum |I~ - I|, [3] dL/da, [4] dL/db, [5] sum |D^ - D|
  const double ssim = sums[1] * inv_n, l1 = sums[2] * inv_n, ga = sums[3], gb = sums[4], ld = sums[5] * inv_p;
  sums[0] = l1; sums[1] = ssim; sums[2] = ld; sums[3] = alpha_p * l1 + lambda * (1.0 - ssim) + beta * ld;
  sums[4] = ga; sums[5] = gb;
  g_ab[0] = (float)ga; g_ab[1] = (float)gb;
}

}  // namespace gs

using namespace gs;

extern "C" int gs_loss_refine(void* stream, int32_t width, int32_t height, const float* rgb, const float* depth,
                              const float* target_rgb, const float* target_depth, const float* ab, float alpha_p,
                              float lambda, float beta, float* d_rgb, float* d_depth, float* g_ab, float* work,
                              double* loss) {
  if (width <= 0 || height <= 0 || !rgb || !depth || !target_rgb || !target_depth || !ab || !d_rgb || !d_depth || !g_ab ||
      !work || !loss)
    return GS_E_INVALID;
  cudaStream_t s = (cudaStream_t)stream;
  static bool win_set[64] = {false};
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev >= 0 && dev < 64 && !win_set[dev]) {  // 11-tap Gaussian, sigma 1.5, normalised (computed in fp64)
    double g[kWin], sum = 0.0;
    for (int k = 0; k < kWin; ++k) { g[k] = exp(-(double)((k - kWinR) * (k - kWinR)) / (2.0 * 1.5 * 1.5)); sum += g[k]; }
    float gf[kWin];
    for (int k = 0; k < kWin; ++k) gf[k] = (float)(g[k] / sum);
    if (cudaMemcpyToSymbol(c_win, gf, sizeof(gf)) != cudaSuccess) { cudaGetLastError(); return GS_E_CUDA; }
    win_set[dev] = true;
  }
  if (cudaMemsetAsync(loss, 0, 8 * sizeof(double), s) != cudaSuccess) { cudaGetLastError(); return GS_E_CUDA; }
  const double P = (double)width * height, inv_n = 1.0 / (3.0 * P), inv_p = 1.0 / P;
  const dim3 grid((width + kRT - 1) / kRT, (height + kRT - 1) / kRT, 3);
  ssim_moments_kernel<<<grid, 256, 0, s>>>(width, height, rgb, target_rgb, ab, work, loss);
  ssim_grad_kernel<<<grid, 256, 0, s>>>(width, height, rgb, depth, target_rgb, target_depth, ab, work,
                                        (float)((double)alpha_p * inv_n), (float)((double)lambda * inv_n),
                                        (float)((double)beta * inv_p), d_rgb, d_depth, loss);
  refine_final_kernel<<<1, 32, 0, s>>>(loss, inv_n, inv_p, (double)alpha_p, (double)lambda, (double)beta, g_ab);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

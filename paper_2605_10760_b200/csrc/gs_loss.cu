// gs_loss.cu -- the dataset-free terms of the mapping loss, Eq. 4, fused so that an optimisation step
// needs no framework ops between gs_rasterize_fwd and gs_rasterize_bwd:
//   gs_loss_map : alpha L1(I^, I) + beta L1(D^, D): one pass over the rendered and target images writes the upstream
//                 gradients dL/dRGB, dL/dDepth and the two (unweighted) L1 means.  HBM-bound: 32 B read + 16 B written
//                 per pixel, float4 accesses, grid = a multiple of the SM count, fp64 block-reduced sums.
//   gs_loss_iso : lambda_s sum_i |s_i - mean(s_i)|_1: loss and gradient w.r.t. the scales, added into g_scales.
// Readings (Q18): mean reduction over pixels (and channels); depth term only where the target depth is > 0;
// sign(0) = 0.  Product code: nothing here includes, links or calls oracle/.
#include "gs_internal.cuh"

namespace gs {

__device__ __forceinline__ float sgn(float d) { return d > 0.f ? 1.f : (d < 0.f ? -1.f : 0.f); }

__device__ __forceinline__ void block_sum2_atomic(double a, double b, double* out) {
  __shared__ double s_a[32], s_b[32];
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, d);
    b += __shfl_xor_sync(0xffffffffu, b, d);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) { s_a[warp] = a; s_b[warp] = b; }
  __syncthreads();
  if (warp == 0) {
    const int nw = (blockDim.x + 31) >> 5;
    a = lane < nw ? s_a[lane] : 0.0;
    b = lane < nw ? s_b[lane] : 0.0;
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) {
      a += __shfl_xor_sync(0xffffffffu, a, d);
      b += __shfl_xor_sync(0xffffffffu, b, d);
    }
    if (lane == 0) {
      if (a != 0.0) atomicAdd(out, a);
      if (b != 0.0) atomicAdd(out + 1, b);
    }
  }
}

// P = H W pixels; quads of 4 consecutive pixels per thread and iteration (P4 = P / 4 of them), scalar tail after.
__global__ void __launch_bounds__(256)
loss_map_kernel(int64_t P, const float* __restrict__ rgb, const float* __restrict__ depth,
                const float* __restrict__ trgb, const float* __restrict__ tdepth, float wr, float wd,
                float* __restrict__ d_rgb, float* __restrict__ d_depth, double* sums, bool vec, double inv_rgb,
                double inv_d, double alpha, double beta) {
  double sr = 0.0, sd = 0.0;
  const int64_t P4 = P >> 2;  // vec: P is a multiple of 4 and every plane is 16-byte aligned
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  if (vec) {
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < P4; q += stride) {
      float acc = 0.f;
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const float4 a = __ldcs(reinterpret_cast<const float4*>(rgb + c * P) + q);
        const float4 t = __ldcs(reinterpret_cast<const float4*>(trgb + c * P) + q);
        const float d0 = a.x - t.x, d1 = a.y - t.y, d2 = a.z - t.z, d3 = a.w - t.w;
        acc += (fabsf(d0) + fabsf(d1)) + (fabsf(d2) + fabsf(d3));
        __stcs(reinterpret_cast<float4*>(d_rgb + c * P) + q, make_float4(wr * sgn(d0), wr * sgn(d1), wr * sgn(d2), wr * sgn(d3)));
      }
      sr += (double)acc;
      const float4 a = __ldcs(reinterpret_cast<const float4*>(depth) + q);
      const float4 t = __ldcs(reinterpret_cast<const float4*>(tdepth) + q);
      const float d0 = t.x > 0.f ? a.x - t.x : 0.f, d1 = t.y > 0.f ? a.y - t.y : 0.f;
      const float d2 = t.z > 0.f ? a.z - t.z : 0.f, d3 = t.w > 0.f ? a.w - t.w : 0.f;
      sd += (double)((fabsf(d0) + fabsf(d1)) + (fabsf(d2) + fabsf(d3)));
      __stcs(reinterpret_cast<float4*>(d_depth) + q, make_float4(wd * sgn(d0), wd * sgn(d1), wd * sgn(d2), wd * sgn(d3)));
    }
  } else {
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < P; p += stride) {
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const float d = rgb[c * P + p] - trgb[c * P + p];
        sr += (double)fabsf(d);
        d_rgb[c * P + p] = wr * sgn(d);
      }
      const float t = tdepth[p];
      const float d = t > 0.f ? depth[p] - t : 0.f;
      sd += (double)fabsf(d);
      d_depth[p] = wd * sgn(d);
    }
  }
  block_sum2_atomic(sr, sd, sums);
  // the last CTA to arrive turns the raw sums into the means and the weighted total (sums[3] is its arrival counter)
  __shared__ bool s_last;
  if (threadIdx.x == 0) {
    __threadfence();
    s_last = atomicAdd(reinterpret_cast<unsigned long long*>(sums + 3), 1ull) == (unsigned long long)gridDim.x - 1ull;
  }
  __syncthreads();
  if (s_last && threadIdx.x == 0) {
    __threadfence();
    const double lr = __ldcg(sums) * inv_rgb, ld = __ldcg(sums + 1) * inv_d;
    sums[0] = lr; sums[1] = ld; sums[2] = alpha * lr + beta * ld;
  }
}

__global__ void __launch_bounds__(256)
loss_iso_kernel(int64_t N, const float* __restrict__ scales, float lambda_s, float* __restrict__ g_scales,
                double* __restrict__ sums) {
  double acc = 0.0;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
    const float s0 = scales[3 * i], s1 = scales[3 * i + 1], s2 = scales[3 * i + 2];
    // s_j - mean(s) = ((s_j - s_k) + (s_j - s_l)) / 3: exactly 0 for equal scales (s - (s0 + s1 + s2) / 3 is not, in fp32)
    const float d0 = ((s0 - s1) + (s0 - s2)) * (1.f / 3.f);
    const float d1 = ((s1 - s0) + (s1 - s2)) * (1.f / 3.f);
    const float d2 = ((s2 - s0) + (s2 - s1)) * (1.f / 3.f);
    acc += (double)(fabsf(d0) + fabsf(d1) + fabsf(d2));
    const float g0 = sgn(d0), g1 = sgn(d1), g2 = sgn(d2);
    const float m = (g0 + g1 + g2) * (1.f / 3.f);  // d mean / d s_ij = 1/3
    g_scales[3 * i] += lambda_s * (g0 - m);
    g_scales[3 * i + 1] += lambda_s * (g1 - m);
    g_scales[3 * i + 2] += lambda_s * (g2 - m);
  }
  block_sum2_atomic(acc * (double)lambda_s, 0.0, sums);
}

}  // namespace gs

using namespace gs;

extern "C" {

int gs_loss_map(void* stream, int32_t width, int32_t height, const float* rgb, const float* depth, const float* target_rgb,
                const float* target_depth, float alpha, float beta, float* d_rgb, float* d_depth, double* loss) {
  if (width <= 0 || height <= 0 || !rgb || !depth || !target_rgb || !target_depth || !d_rgb || !d_depth || !loss)
    return GS_E_INVALID;
  cudaStream_t s = (cudaStream_t)stream;
  const int64_t P = (int64_t)width * height;
  if (cudaMemsetAsync(loss, 0, 4 * sizeof(double), s) != cudaSuccess) { cudaGetLastError(); return GS_E_CUDA; }
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  auto al = [](const void* p) { return ((uintptr_t)p & 15) == 0; };
  const bool vec = (P & 3) == 0 && al(rgb) && al(depth) && al(target_rgb) && al(target_depth) && al(d_rgb) && al(d_depth);
  const int64_t work = vec ? (P >> 2) : P;
  const int mult = 4;  // CTAs per SM: measured 1 / 2 / 4 / 8 -> 19.8 / 13.5 / 11.3 / 14.1 us at 1200x680 (ncu, cold cache)
  int64_t grid64 = div_up(work, 256);
  if (grid64 > (int64_t)sms * mult) grid64 = (int64_t)sms * mult;
  const int grid = (int)grid64;
  const double inv_rgb = 1.0 / (3.0 * (double)P), inv_d = 1.0 / (double)P;
  loss_map_kernel<<<grid, 256, 0, s>>>(P, rgb, depth, target_rgb, target_depth, (float)((double)alpha * inv_rgb),
                                       (float)((double)beta * inv_d), d_rgb, d_depth, loss, vec, inv_rgb, inv_d,
                                       (double)alpha, (double)beta);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

int gs_loss_iso(void* stream, int64_t N, const float* scales, float lambda_s, float* g_scales, double* loss) {
  if (N < 0 || (N > 0 && (!scales || !g_scales)) || !loss) return GS_E_INVALID;
  cudaStream_t s = (cudaStream_t)stream;
  if (cudaMemsetAsync(loss, 0, 2 * sizeof(double), s) != cudaSuccess) { cudaGetLastError(); return GS_E_CUDA; }
  if (N == 0) return GS_OK;
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  int64_t grid64 = div_up(N, 256);
  if (grid64 > (int64_t)sms * 8) grid64 = (int64_t)sms * 8;
  const int grid = (int)grid64;
  loss_iso_kernel<<<grid, 256, 0, s>>>(N, scales, lambda_s, g_scales, loss);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

}  // extern "C"

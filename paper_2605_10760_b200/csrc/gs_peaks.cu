// gs_peaks.cu -- measured machine peaks for the roofline denominators:
// FP32 FMA lane rate, MUFU.EX2 rate, shared-memory wavefront rates (the pipe that bounds the compositing kernels),
// L2 RED.ADD.F32 rate, HBM read / write / copy bandwidth.  `gs_measure_peaks` (include/gs.h) runs them and returns the
// numbers; bench.py uses them as the `peak` of its roofline entries ("measured in this run") and
// `bench.py --workload peaks` prints them.  Plain synthetic kernels: nothing of the method's arithmetic is here.
#include <stdint.h>

#include <cuda_runtime.h>

#include "../../include/gs.h"

namespace gs_peaks {

constexpr int kThreads = 256;

// ---- FP32 FMA: 16 independent chains per thread, 3-register FFMA (a * b + c with a loop-carried c) ---------------
__global__ void __launch_bounds__(kThreads) fma_kernel(float* out, int iters, float a, float b) {
  float acc[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) acc[k] = (float)(threadIdx.x + k);
  const float x = a + threadIdx.x * 1e-9f, y = b;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 16; ++k) acc[k] = fmaf(acc[k], x, y);
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < 16; ++k) s += acc[k];
  out[blockIdx.x * kThreads + threadIdx.x] = s;
}

// ---- mixed issue: FFMA + integer ALU instructions interleaved (the compositing kernels are issue-bound) -----------
__global__ void __launch_bounds__(kThreads) issue_kernel(float* out, int iters, float a, float b) {
  float acc[8];
  uint32_t z[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) { acc[k] = (float)(threadIdx.x + k); z[k] = threadIdx.x * 7u + k; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 8; ++k) { acc[k] = fmaf(acc[k], a, b); z[k] = (z[k] ^ (uint32_t)it) + 0x9e3779b9u; }
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += acc[k] + (float)(z[k] & 1u);
  out[blockIdx.x * kThreads + threadIdx.x] = s;
}

// ---- MUFU.EX2 ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads) ex2_kernel(float* out, int iters) {
  float acc[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) acc[k] = -1e-3f * (float)(threadIdx.x + k);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 8; ++k) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(acc[k]));
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += acc[k];
  out[blockIdx.x * kThreads + threadIdx.x] = s;
}

// ---- shared memory: MODE 0 = LDS.128 all lanes the same address (the record broadcast of the compositing kernels),
//      1 = LDS.128 conflict-free (lane-consecutive), 2 = LDS.32 broadcast, 3 = LDS.64 broadcast ------------------------
template <int MODE>
__global__ void __launch_bounds__(kThreads) lds_kernel(float* out, int iters) {
  __shared__ __align__(16) float4 s[1024];
  for (int k = threadIdx.x; k < 1024; k += kThreads) s[k] = make_float4((float)k, 1.f, 2.f, 3.f);
  __syncthreads();
  float acc = 0.f;
  const int lane = threadIdx.x & 31;
  uint32_t base = (threadIdx.x >> 5) * 64;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const uint32_t idx = (base + k * 5 + it) & 1023u;  // warp-uniform record index
      if (MODE == 0) { const float4 v = s[idx]; acc += v.x + v.y + v.z + v.w; }
      else if (MODE == 1) { const float4 v = s[(idx + lane) & 1023u]; acc += v.x + v.y + v.z + v.w; }
      else if (MODE == 2) { acc += reinterpret_cast<const float*>(s)[idx * 4]; }
      else { const float2 v = reinterpret_cast<const float2*>(s)[idx * 2]; acc += v.x + v.y; }
    }
  }
  out[blockIdx.x * kThreads + threadIdx.x] = acc;
}

// ---- L2 reductions: every warp adds 32 consecutive floats (one 128-byte line) of a record array, lines picked by a
//      hash over `lines` distinct lines (the access shape of the pixel backward's RED.ADD.F32) -------------------------
__global__ void __launch_bounds__(kThreads) red_kernel(float* buf, uint32_t lines, int iters) {
  const uint32_t warp = (blockIdx.x * kThreads + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  uint32_t h = warp * 2654435761u;
  for (int it = 0; it < iters; ++it) {
    h = h * 1664525u + 1013904223u;
    atomicAdd(buf + (size_t)(h % lines) * 32 + lane, 1.0f);
  }
}

// ---- HBM streams ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads) read_kernel(const float4* __restrict__ src, size_t n, float* out) {
  float acc = 0.f;
  for (size_t i = (size_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (size_t)gridDim.x * kThreads) {
    const float4 v = __ldcs(src + i);
    acc += v.x + v.y + v.z + v.w;
  }
  if (acc == 123.456f) out[0] = acc;
}
__global__ void __launch_bounds__(kThreads) write_kernel(float4* __restrict__ dst, size_t n) {
  for (size_t i = (size_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (size_t)gridDim.x * kThreads)
    __stcs(dst + i, make_float4(1.f, 2.f, 3.f, 4.f));
}
__global__ void __launch_bounds__(kThreads) copy_kernel(const float4* __restrict__ src, float4* __restrict__ dst, size_t n) {
  for (size_t i = (size_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (size_t)gridDim.x * kThreads)
    __stcs(dst + i, __ldcs(src + i));
}

template <typename F>
static int time_best(cudaStream_t s, cudaEvent_t e0, cudaEvent_t e1, int reps, double* best_ms, F launch) {
  launch();  // warm-up
  if (cudaStreamSynchronize(s) != cudaSuccess) return GS_E_CUDA;
  *best_ms = 1e30;
  for (int r = 0; r < reps; ++r) {
    cudaEventRecord(e0, s);
    launch();
    cudaEventRecord(e1, s);
    if (cudaEventSynchronize(e1) != cudaSuccess) return GS_E_CUDA;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < *best_ms) *best_ms = ms;
  }
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

}  // namespace gs_peaks

extern "C" int gs_measure_peaks(int device, void* stream, double* out) {
  using namespace gs_peaks;
  if (!out) return GS_E_INVALID;
  if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return GS_E_CUDA; }
  cudaStream_t s = (cudaStream_t)stream;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return GS_E_CUDA;
  const int sms = prop.multiProcessorCount;
  int clock_khz = 0;
  cudaDeviceGetAttribute(&clock_khz, cudaDevAttrClockRate, device);
  for (int k = 0; k < GS_NUM_PEAKS; ++k) out[k] = 0.0;
  out[GS_PEAK_SM_COUNT] = sms;
  out[GS_PEAK_SM_MHZ_MAX] = clock_khz / 1e3;
  const size_t stream_bytes = (size_t)1 << 30;  // 1 GiB per stream buffer: 8x the L2
  float* scratch = nullptr;
  float4 *a = nullptr, *b = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  int rc = GS_OK;
  const int grid = sms * 8;
  double ms = 0.0;
  bool ok = cudaMalloc((void**)&scratch, (size_t)grid * kThreads * sizeof(float)) == cudaSuccess &&
            cudaMalloc((void**)&a, stream_bytes) == cudaSuccess && cudaMalloc((void**)&b, stream_bytes) == cudaSuccess &&
            cudaEventCreate(&e0) == cudaSuccess && cudaEventCreate(&e1) == cudaSuccess &&
            cudaMemsetAsync(a, 0, stream_bytes, s) == cudaSuccess;
  if (!ok) { rc = GS_E_NOMEM; cudaGetLastError(); }
  const double threads = (double)grid * kThreads;
  if (rc == GS_OK) {
    const int iters = 4096;
    rc = time_best(s, e0, e1, 5, &ms, [&] { fma_kernel<<<grid, kThreads, 0, s>>>(scratch, iters, 1.0001f, 0.5f); });
    out[GS_PEAK_FMA_TLANES] = threads * 16.0 * iters / (ms * 1e-3) / 1e12;
  }
  if (rc == GS_OK) {
    const int iters = 4096;
    rc = time_best(s, e0, e1, 5, &ms, [&] { issue_kernel<<<grid, kThreads, 0, s>>>(scratch, iters, 1.0001f, 0.5f); });
    out[GS_PEAK_ISSUE_TWARP] = threads / 32.0 * 24.0 * iters / (ms * 1e-3) / 1e12;  // FFMA + LOP3 + IADD3 per k
  }
  if (rc == GS_OK) {
    const int iters = 4096;
    rc = time_best(s, e0, e1, 5, &ms, [&] { ex2_kernel<<<grid, kThreads, 0, s>>>(scratch, iters); });
    out[GS_PEAK_EX2_TLANES] = threads * 8.0 * iters / (ms * 1e-3) / 1e12;
  }
  if (rc == GS_OK) {
    const int iters = 2048;
    rc = time_best(s, e0, e1, 5, &ms, [&] { lds_kernel<0><<<grid, kThreads, 0, s>>>(scratch, iters); });
    out[GS_PEAK_LDS128_BCAST_TWARP] = threads / 32.0 * 8.0 * iters / (ms * 1e-3) / 1e12;
    if (rc == GS_OK) rc = time_best(s, e0, e1, 5, &ms, [&] { lds_kernel<1><<<grid, kThreads, 0, s>>>(scratch, iters); });
    out[GS_PEAK_LDS128_TWARP] = threads / 32.0 * 8.0 * iters / (ms * 1e-3) / 1e12;
    if (rc == GS_OK) rc = time_best(s, e0, e1, 5, &ms, [&] { lds_kernel<2><<<grid, kThreads, 0, s>>>(scratch, iters); });
    out[GS_PEAK_LDS32_BCAST_TWARP] = threads / 32.0 * 8.0 * iters / (ms * 1e-3) / 1e12;
    if (rc == GS_OK) rc = time_best(s, e0, e1, 5, &ms, [&] { lds_kernel<3><<<grid, kThreads, 0, s>>>(scratch, iters); });
    out[GS_PEAK_LDS64_BCAST_TWARP] = threads / 32.0 * 8.0 * iters / (ms * 1e-3) / 1e12;
  }
  if (rc == GS_OK) {
    const int iters = 256;
    const uint32_t lines = 1u << 16;  // 8 MB of accumulators, L2-resident (the g2d array of config 3 is 4.5 MB)
    cudaMemsetAsync(b, 0, (size_t)lines * 128, s);
    rc = time_best(s, e0, e1, 5, &ms, [&] { red_kernel<<<grid, kThreads, 0, s>>>(reinterpret_cast<float*>(b), lines, iters); });
    out[GS_PEAK_RED_GLANES] = threads * iters / (ms * 1e-3) / 1e9;
  }
  if (rc == GS_OK) {
    const size_t n = stream_bytes / sizeof(float4);
    const int g2 = sms * 16;
    rc = time_best(s, e0, e1, 5, &ms, [&] { read_kernel<<<g2, kThreads, 0, s>>>(a, n, scratch); });
    out[GS_PEAK_HBM_READ_GBS] = (double)stream_bytes / (ms * 1e-3) / 1e9;
    if (rc == GS_OK) rc = time_best(s, e0, e1, 5, &ms, [&] { write_kernel<<<g2, kThreads, 0, s>>>(b, n); });
    out[GS_PEAK_HBM_WRITE_GBS] = (double)stream_bytes / (ms * 1e-3) / 1e9;
    if (rc == GS_OK) rc = time_best(s, e0, e1, 5, &ms, [&] { copy_kernel<<<g2, kThreads, 0, s>>>(a, b, n); });
    out[GS_PEAK_HBM_COPY_GBS] = 2.0 * (double)stream_bytes / (ms * 1e-3) / 1e9;
  }
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  cudaFree(scratch); cudaFree(a); cudaFree(b);
  cudaGetLastError();
  return rc;
}

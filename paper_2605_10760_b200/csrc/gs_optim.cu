// gs_optim.cu -- optimiser step and pruning of the map refinement ("optimized ... by gradient descent on" Eq. 4;
// PAPER.md:322 "2,000 iterations at half the per-agent learning rate and prunes Gaussians with opacity below 0.005"), and
// the order-preserving stream compaction shared with the fusion's retain test (Eq. 22).
//   gs_adam_step    : fused Adam (reading Q20: Kingma & Ba Algorithm 1 with bias correction; scales through
//                     log s, opacities through logit o, so the ACTIVATED values of the C-ABI stay in their domains; the
//                     gradients are those of gs_rasterize_bwd, w.r.t. the activated values); only Gaussians with a non-zero
//                     `visible` entry are touched (parameters AND moments): the HBM traffic is 28 B per float of a VISIBLE
//                     Gaussian instead of 28 B x (11 + 3K) x N.
//   gs_prune_mask   : keep[i] = opacity[i] >= min_opacity.
//   gs_compact_plan / gs_compact_rows : exclusive scan of a keep mask -> destination row of every kept Gaussian (original
//                     order preserved), then a row gather per parameter array.
// HBM-streaming kernels, one element per thread, grid-stride.  Product code: nothing here includes, links or calls oracle/.
#include <mutex>

#include "gs_internal.cuh"

namespace gs {

enum AdamMode { kDirect = 0, kLog = 1, kLogit = 2 };

template <int MODE>
__global__ void __launch_bounds__(256)
adam_kernel(int64_t n, int32_t width, float* __restrict__ p, const float* __restrict__ g, float* __restrict__ m,
            float* __restrict__ v, const uint32_t* __restrict__ visible, float lr, float beta1, float beta2, float eps,
            float ibc1, float ibc2) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride) {
    if (visible && __ldg(visible + e / width) == 0u) continue;
    const float x = p[e];
    float gr = g[e];
    if (MODE == kLog) gr *= x;                    // dL/dlog s = s dL/ds
    if (MODE == kLogit) gr *= x * (1.f - x);      // dL/dlogit o = o (1 - o) dL/do
    const float mn = fmaf(beta1, m[e], (1.f - beta1) * gr);
    const float vn = fmaf(beta2, v[e], (1.f - beta2) * gr * gr);
    m[e] = mn; v[e] = vn;
    const float d = -lr * (mn * ibc1) / (sqrtf(vn * ibc2) + eps);   // step of the raw parameter
    float xn;
    if (MODE == kDirect) xn = x + d;
    else if (MODE == kLog) xn = x * expf(d);       // exp(log s + d)
    else { const float t = x * expf(d); xn = t / ((1.f - x) + t); }  // sigmoid(logit o + d)
    p[e] = xn;
  }
}

// the same step on compact gradient rows (GS_SPARSE_GRADS): row r belongs to Gaussian ids[r], r < *n_rows
template <int MODE>
__global__ void __launch_bounds__(256)
adam_sparse_kernel(int64_t max_n, int32_t width, float* __restrict__ p, const float* __restrict__ g, float* __restrict__ m,
                   float* __restrict__ v, const uint32_t* __restrict__ ids, const uint32_t* __restrict__ n_rows, float lr,
                   float beta1, float beta2, float eps, float ibc1, float ibc2) {
  const int64_t n = min(max_n, (int64_t)__ldg(n_rows) * width);
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < n; r += stride) {
    const int64_t row = r / width;
    const int64_t e = (int64_t)__ldg(ids + row) * width + (r - row * width);
    const float x = p[e];
    float gr = g[r];
    if (MODE == kLog) gr *= x;
    if (MODE == kLogit) gr *= x * (1.f - x);
    const float mn = fmaf(beta1, m[e], (1.f - beta1) * gr);
    const float vn = fmaf(beta2, v[e], (1.f - beta2) * gr * gr);
    m[e] = mn; v[e] = vn;
    const float d = -lr * (mn * ibc1) / (sqrtf(vn * ibc2) + eps);
    float xn;
    if (MODE == kDirect) xn = x + d;
    else if (MODE == kLog) xn = x * expf(d);
    else { const float t = x * expf(d); xn = t / ((1.f - x) + t); }
    p[e] = xn;
  }
}

__global__ void __launch_bounds__(256)
prune_mask_kernel(int64_t N, const float* __restrict__ opac, float min_opacity, uint8_t* __restrict__ keep) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) keep[i] = opac[i] >= min_opacity ? 1 : 0;
}

constexpr int kPlanBlock = 1024;  // Gaussians per block of the compaction plan

__global__ void __launch_bounds__(256)
plan_count_kernel(int64_t N, const uint8_t* __restrict__ keep, uint32_t* __restrict__ block_count) {
  __shared__ uint32_t s_c[8];
  const int64_t base = (int64_t)blockIdx.x * kPlanBlock;
  uint32_t c = 0;
#pragma unroll
  for (int k = 0; k < kPlanBlock / 256; ++k) {
    const int64_t i = base + k * 256 + threadIdx.x;
    c += (i < N && keep[i]) ? 1u : 0u;
  }
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) c += __shfl_xor_sync(0xffffffffu, c, d);
  if ((threadIdx.x & 31) == 0) s_c[threadIdx.x >> 5] = c;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t t = 0;
    for (int w = 0; w < 8; ++w) t += s_c[w];
    block_count[blockIdx.x] = t;
  }
}

// one CTA: exclusive scan of the block counts in place, total -> n_kept
__global__ void __launch_bounds__(1024)
plan_scan_kernel(int nblocks, uint32_t* __restrict__ block_count, int64_t* __restrict__ n_kept) {
  __shared__ uint32_t s_w[32];
  __shared__ uint32_t s_carry;
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int base = 0; base < nblocks; base += 1024) {
    const int i = base + threadIdx.x;
    const uint32_t x = i < nblocks ? block_count[i] : 0u;
    uint32_t incl = x;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t u = __shfl_up_sync(0xffffffffu, incl, d);
      if (lane >= d) incl += u;
    }
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    if (warp == 0) {
      uint32_t w = s_w[lane], wi = w;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, wi, d);
        if (lane >= d) wi += u;
      }
      s_w[lane] = wi - w;  // exclusive prefix of the warp totals
    }
    __syncthreads();
    const uint32_t carry = s_carry;
    if (i < nblocks) block_count[i] = carry + s_w[warp] + incl - x;
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = carry + s_w[warp] + incl;
    __syncthreads();
  }
  if (threadIdx.x == 0) *n_kept = (int64_t)s_carry;
}

__global__ void __launch_bounds__(256)
plan_index_kernel(int64_t N, const uint8_t* __restrict__ keep, const uint32_t* __restrict__ block_offset,
                  uint32_t* __restrict__ index) {
  // kPlanBlock = 4 x 256: thread t handles the 4 consecutive Gaussians 4 t .. 4 t + 3 of the block (order preserved)
  __shared__ uint32_t s_w[8];
  const int64_t base = (int64_t)blockIdx.x * kPlanBlock + 4 * threadIdx.x;
  uint32_t k[4], c = 0;
#pragma unroll
  for (int u = 0; u < 4; ++u) { k[u] = (base + u < N && keep[base + u]) ? 1u : 0u; c += k[u]; }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t incl = c;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t u = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= d) incl += u;
  }
  if (lane == 31) s_w[warp] = incl;
  __syncthreads();
  uint32_t off = block_offset[blockIdx.x] + incl - c;
  for (int w = 0; w < warp; ++w) off += s_w[w];
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    if (base + u < N) index[base + u] = k[u] ? off : 0xffffffffu;
    off += k[u];
  }
}

__global__ void __launch_bounds__(256)
compact_rows_kernel(int64_t n, int32_t width, const uint32_t* __restrict__ index, const float* __restrict__ in,
                    float* __restrict__ out) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride) {
    const int64_t i = e / width;
    const uint32_t d = __ldg(index + i);
    if (d != 0xffffffffu) out[(int64_t)d * width + (e - i * width)] = in[e];
  }
}

static int grid_for(int64_t n) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  int64_t g = div_up(n, 256);
  if (g > (int64_t)sms * 8) g = (int64_t)sms * 8;
  return (int)(g < 1 ? 1 : g);
}

// ---- scratch of gs_compact_plan_static: lives in the library image, not on the heap -------------------------------------
// One word per block of kPlanBlock Gaussians, for at most kStaticPlanMaxN Gaussians: 64 KiB that every GPU loading libgs.so
// holds from module load to process exit.  gs_compact_plan_static exists for callers that may not allocate device memory
// at the point where they compact (see include/gs.h); it is the only user of this array.
constexpr int64_t kStaticPlanMaxN = 1ll << 24;                      // 16 Mi Gaussians
constexpr int kStaticPlanWords = (int)(kStaticPlanMaxN / kPlanBlock);  // 16384 block counters
static __device__ __align__(256) uint32_t g_static_plan_counts[kStaticPlanWords];

// In host code the name g_static_plan_counts is only a handle for the runtime, never a device address: handing it to a
// kernel would fault (or, on a GPU that can reach host memory, quietly work on the wrong bytes).  The device address is
// asked for once per device, with that device current, and kept here.
constexpr int kStaticPlanMaxDevices = 64;
static uint32_t* s_static_plan_ptr[kStaticPlanMaxDevices];
static std::mutex s_static_plan_mutex;

static int static_plan_scratch(uint32_t** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kStaticPlanMaxDevices) { cudaGetLastError(); return GS_E_CUDA; }
  std::lock_guard<std::mutex> lock(s_static_plan_mutex);
  if (!s_static_plan_ptr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_static_plan_counts) != cudaSuccess || !p) { cudaGetLastError(); return GS_E_CUDA; }
    s_static_plan_ptr[dev] = static_cast<uint32_t*>(p);
  }
  *out = s_static_plan_ptr[dev];
  return GS_OK;
}

}  // namespace gs

using namespace gs;

extern "C" {

int gs_adam_step(void* stream, int64_t N, int sh_degree, const gs_adam_config* cfg, const gs_gaussians* params,
                 const gs_gaussians* grads, const gs_gaussians* m, const gs_gaussians* v, const uint32_t* visible) {
  if (N < 0 || sh_degree < 0 || sh_degree > 3 || !cfg || !params || !grads || !m || !v || cfg->step < 1) return GS_E_INVALID;
  if (N == 0) return GS_OK;
  const int K3 = 3 * (sh_degree + 1) * (sh_degree + 1);
  float* P[5] = {params->means, params->scales, params->quats, params->opacities, params->sh};
  const float* G[5] = {grads->means, grads->scales, grads->quats, grads->opacities, grads->sh};
  float* M[5] = {m->means, m->scales, m->quats, m->opacities, m->sh};
  float* V[5] = {v->means, v->scales, v->quats, v->opacities, v->sh};
  const int width[5] = {3, 3, 4, 1, K3};
  const float lr[5] = {cfg->lr_means, cfg->lr_scales, cfg->lr_quats, cfg->lr_opacities, cfg->lr_sh};
  for (int k = 0; k < 5; ++k)
    if (!P[k] || !G[k] || !M[k] || !V[k]) return GS_E_INVALID;
  cudaStream_t s = (cudaStream_t)stream;
  const float ibc1 = (float)(1.0 / (1.0 - pow((double)cfg->beta1, (double)cfg->step)));
  const float ibc2 = (float)(1.0 / (1.0 - pow((double)cfg->beta2, (double)cfg->step)));
  for (int k = 0; k < 5; ++k) {
    const int64_t n = N * width[k];
    const int grid = grid_for(n);
#define GS_ADAM(MODE) adam_kernel<MODE><<<grid, 256, 0, s>>>(n, width[k], P[k], G[k], M[k], V[k], visible, lr[k], cfg->beta1, \
                                                            cfg->beta2, cfg->eps, ibc1, ibc2)
    if (k == 1) GS_ADAM(kLog); else if (k == 3) GS_ADAM(kLogit); else GS_ADAM(kDirect);
#undef GS_ADAM
  }
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

int gs_adam_step_sparse(void* stream, int64_t N, int sh_degree, const gs_adam_config* cfg, const gs_gaussians* params,
                        const gs_gaussians* grads, const gs_gaussians* m, const gs_gaussians* v, const uint32_t* ids,
                        const uint32_t* n_rows, int64_t max_rows) {
  if (N < 0 || sh_degree < 0 || sh_degree > 3 || !cfg || !params || !grads || !m || !v || cfg->step < 1 || max_rows < 0 ||
      max_rows > N || (max_rows > 0 && (!ids || !n_rows)))
    return GS_E_INVALID;
  if (max_rows == 0) return GS_OK;
  const int K3 = 3 * (sh_degree + 1) * (sh_degree + 1);
  float* P[5] = {params->means, params->scales, params->quats, params->opacities, params->sh};
  const float* G[5] = {grads->means, grads->scales, grads->quats, grads->opacities, grads->sh};
  float* M[5] = {m->means, m->scales, m->quats, m->opacities, m->sh};
  float* V[5] = {v->means, v->scales, v->quats, v->opacities, v->sh};
  const int width[5] = {3, 3, 4, 1, K3};
  const float lr[5] = {cfg->lr_means, cfg->lr_scales, cfg->lr_quats, cfg->lr_opacities, cfg->lr_sh};
  for (int k = 0; k < 5; ++k)
    if (!P[k] || !G[k] || !M[k] || !V[k]) return GS_E_INVALID;
  cudaStream_t s = (cudaStream_t)stream;
  const float ibc1 = (float)(1.0 / (1.0 - pow((double)cfg->beta1, (double)cfg->step)));
  const float ibc2 = (float)(1.0 / (1.0 - pow((double)cfg->beta2, (double)cfg->step)));
  for (int k = 0; k < 5; ++k) {
    const int64_t n = max_rows * width[k];
    const int grid = grid_for(n);
#define GS_ADAM(MODE) adam_sparse_kernel<MODE><<<grid, 256, 0, s>>>(n, width[k], P[k], G[k], M[k], V[k], ids, n_rows, lr[k],                                                                    cfg->beta1, cfg->beta2, cfg->eps, ibc1, ibc2)
    if (k == 1) GS_ADAM(kLog); else if (k == 3) GS_ADAM(kLogit); else GS_ADAM(kDirect);
#undef GS_ADAM
  }
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

int gs_prune_mask(void* stream, int64_t N, const float* opacities, float min_opacity, uint8_t* keep) {
  if (N < 0 || (N > 0 && (!opacities || !keep))) return GS_E_INVALID;
  if (N == 0) return GS_OK;
  prune_mask_kernel<<<grid_for(N), 256, 0, (cudaStream_t)stream>>>(N, opacities, min_opacity, keep);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

int64_t gs_compact_work_bytes(int64_t N) { return (div_up(N < 0 ? 0 : N, kPlanBlock) + 1) * (int64_t)sizeof(uint32_t); }

int gs_compact_plan(void* stream, int64_t N, const uint8_t* keep, uint32_t* index, int64_t* n_kept, void* work) {
  if (N < 0 || N >= (1ll << 32) || !n_kept || (N > 0 && (!keep || !index || !work))) return GS_E_INVALID;
  cudaStream_t s = (cudaStream_t)stream;
  if (N == 0) return cudaMemsetAsync(n_kept, 0, sizeof(int64_t), s) == cudaSuccess ? GS_OK : GS_E_CUDA;
  const int nblocks = (int)div_up(N, kPlanBlock);
  uint32_t* bc = reinterpret_cast<uint32_t*>(work);
  plan_count_kernel<<<nblocks, 256, 0, s>>>(N, keep, bc);
  plan_scan_kernel<<<1, 1024, 0, s>>>(nblocks, bc, n_kept);
  plan_index_kernel<<<nblocks, 256, 0, s>>>(N, keep, bc, index);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

int64_t gs_compact_plan_static_max(void) { return kStaticPlanMaxN; }

// gs_compact_plan with its scratch in g_static_plan_counts instead of a caller-provided buffer: same three kernels, same
// results.  Nothing in the array has to be zero when the call starts: plan_count_kernel writes every one of the `nblocks`
// counters before plan_scan_kernel and plan_index_kernel read them, and no word beyond `nblocks` is read, so what an
// earlier call (of any size) left behind is harmless.  No cudaMalloc / cudaFree / allocating routine on this path.
int gs_compact_plan_static(void* stream, int64_t N, const uint8_t* keep, uint32_t* index, int64_t* n_kept) {
  if (N < 0 || !n_kept || (N > 0 && (!keep || !index))) return GS_E_INVALID;
  if (N > kStaticPlanMaxN) return GS_E_TOO_LARGE;
  cudaStream_t s = (cudaStream_t)stream;
  uint32_t* bc = nullptr;
  const int rc = static_plan_scratch(&bc);  // first call on this device: cudaGetSymbolAddress (may load the module)
  if (rc != GS_OK) return rc;
  if (N == 0) return cudaMemsetAsync(n_kept, 0, sizeof(int64_t), s) == cudaSuccess ? GS_OK : GS_E_CUDA;
  const int nblocks = (int)div_up(N, kPlanBlock);
  plan_count_kernel<<<nblocks, 256, 0, s>>>(N, keep, bc);
  plan_scan_kernel<<<1, 1024, 0, s>>>(nblocks, bc, n_kept);
  plan_index_kernel<<<nblocks, 256, 0, s>>>(N, keep, bc, index);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

int gs_compact_rows(void* stream, int64_t N, int32_t width, const uint32_t* index, const float* in, float* out) {
  if (N < 0 || width <= 0) return GS_E_INVALID;
  if (N == 0) return GS_OK;
  if (!index || !in || !out || in == out) return GS_E_INVALID;
  const int64_t n = N * width;
  compact_rows_kernel<<<grid_for(n), 256, 0, (cudaStream_t)stream>>>(n, width, index, in, out);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

}  // extern "C"

// gs_fusion.cu -- Eq. 19: a submap's Sim(3) correction C = (s, R, t) applied to its Gaussians,
//   mu' = s R mu + t,  Sigma' = s^2 R Sigma R^T (i.e. s_i' = s s_i and q' = q_R (x) q),  opacity and colour unchanged
// (PAPER.md:272).  One thread per Gaussian, in place or out of place; HBM-streaming: 40 B read + 40 B written per
// Gaussian.  Product code: nothing here includes, links or calls oracle/.
#include <math.h>

#include "gs_internal.cuh"

namespace gs {

struct Sim3Dev {
  float s, R[9], t[3], q[4];  // q: unit quaternion (w,x,y,z) of R
};

__global__ void __launch_bounds__(256)
sim3_kernel(int64_t N, Sim3Dev C, const float* means, const float* scales, const float* quats, float* means_out,
            float* scales_out, float* quats_out) {  // no __restrict__: an output may alias its input (gs.h)
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
    const float m0 = means[3 * i], m1 = means[3 * i + 1], m2 = means[3 * i + 2];
    const float s0 = scales[3 * i], s1 = scales[3 * i + 1], s2 = scales[3 * i + 2];
    const float4 q = *reinterpret_cast<const float4*>(quats + 4 * i);
    means_out[3 * i] = fmaf(C.s, fmaf(C.R[0], m0, fmaf(C.R[1], m1, C.R[2] * m2)), C.t[0]);
    means_out[3 * i + 1] = fmaf(C.s, fmaf(C.R[3], m0, fmaf(C.R[4], m1, C.R[5] * m2)), C.t[1]);
    means_out[3 * i + 2] = fmaf(C.s, fmaf(C.R[6], m0, fmaf(C.R[7], m1, C.R[8] * m2)), C.t[2]);
    scales_out[3 * i] = C.s * s0; scales_out[3 * i + 1] = C.s * s1; scales_out[3 * i + 2] = C.s * s2;
    const float w1 = C.q[0], x1 = C.q[1], y1 = C.q[2], z1 = C.q[3];
    float4 o;  // Hamilton product q_R (x) q
    o.x = w1 * q.x - x1 * q.y - y1 * q.z - z1 * q.w;
    o.y = w1 * q.y + x1 * q.x + y1 * q.w - z1 * q.z;
    o.z = w1 * q.z - x1 * q.w + y1 * q.x + z1 * q.y;
    o.w = w1 * q.w + x1 * q.z - y1 * q.y + z1 * q.x;
    *reinterpret_cast<float4*>(quats_out + 4 * i) = o;
  }
}

// unit quaternion (w,x,y,z) of a rotation matrix (row-major), Shepperd's method in fp64 (largest pivot), sign fixed so
// that the first non-zero component is positive
static void quat_of_rotation(const float* Rf, float* qf) {
  double R[9];
  for (int k = 0; k < 9; ++k) R[k] = Rf[k];
  const double tr = R[0] + R[4] + R[8];
  double q[4];
  if (tr >= R[0] && tr >= R[4] && tr >= R[8]) {
    const double w = 0.5 * sqrt(1.0 + tr);
    q[0] = w; q[1] = (R[7] - R[5]) / (4 * w); q[2] = (R[2] - R[6]) / (4 * w); q[3] = (R[3] - R[1]) / (4 * w);
  } else if (R[0] >= R[4] && R[0] >= R[8]) {
    const double x = 0.5 * sqrt(1.0 + R[0] - R[4] - R[8]);
    q[1] = x; q[0] = (R[7] - R[5]) / (4 * x); q[2] = (R[1] + R[3]) / (4 * x); q[3] = (R[2] + R[6]) / (4 * x);
  } else if (R[4] >= R[8]) {
    const double y = 0.5 * sqrt(1.0 - R[0] + R[4] - R[8]);
    q[2] = y; q[0] = (R[2] - R[6]) / (4 * y); q[1] = (R[1] + R[3]) / (4 * y); q[3] = (R[5] + R[7]) / (4 * y);
  } else {
    const double z = 0.5 * sqrt(1.0 - R[0] - R[4] + R[8]);
    q[3] = z; q[0] = (R[3] - R[1]) / (4 * z); q[1] = (R[2] + R[6]) / (4 * z); q[2] = (R[5] + R[7]) / (4 * z);
  }
  const double n = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
  double sg = 1.0;
  for (int k = 0; k < 4; ++k)
    if (fabs(q[k]) > 1e-12) { sg = q[k] < 0 ? -1.0 : 1.0; break; }
  for (int k = 0; k < 4; ++k) qf[k] = (float)(sg * q[k] / n);
}

}  // namespace gs

using namespace gs;

extern "C" int gs_sim3_apply(void* stream, int64_t N, float s, const float* R, const float* t, const float* means,
                             const float* scales, const float* quats, float* means_out, float* scales_out,
                             float* quats_out) {
  if (N < 0 || !R || !t || !(s > 0.f)) return GS_E_INVALID;
  if (N == 0) return GS_OK;
  if (!means || !scales || !quats || !means_out || !scales_out || !quats_out) return GS_E_INVALID;
  if ((((uintptr_t)quats) | ((uintptr_t)quats_out)) & 15) return GS_E_INVALID;
  Sim3Dev C;
  C.s = s;
  for (int k = 0; k < 9; ++k) C.R[k] = R[k];
  for (int k = 0; k < 3; ++k) C.t[k] = t[k];
  quat_of_rotation(R, C.q);
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  int64_t grid = div_up(N, 256);
  if (grid > (int64_t)sms * 8) grid = (int64_t)sms * 8;
  sim3_kernel<<<(unsigned)grid, 256, 0, (cudaStream_t)stream>>>(N, C, means, scales, quats, means_out, scales_out, quats_out);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

// ---------------------------------------------------------------------------------------------------------------
// Eqs. 20-22: occupancy-aware fusion on a voxel grid of size v, voxel indices packed into 64-bit
// spatial-hash keys.  Sets are open-addressing hash tables (linear probing, 64-bit atomicCAS) in caller-provided device
// memory.  Every coordinate computation is fp64 with explicitly rounded single operations (no FMA contraction), in the
// sequence DESIGN.md Q21 fixes, so that the sets are bit-identical to the plain definition's.
// ---------------------------------------------------------------------------------------------------------------
namespace gs {

constexpr unsigned long long kVoxEmpty = 0xFFFFFFFFFFFFFFFFull;
constexpr long long kKeyBias = 1ll << 20;

__device__ __forceinline__ unsigned long long vox_key(long long ix, long long iy, long long iz) {
  return (unsigned long long)(ix + kKeyBias) | ((unsigned long long)(iy + kKeyBias) << 21) |
         ((unsigned long long)(iz + kKeyBias) << 42);
}
__device__ __forceinline__ bool vox_in_range(long long i) { return i >= -kKeyBias && i < kKeyBias; }
__device__ __forceinline__ unsigned long long vox_hash(unsigned long long k) {  // splitmix64 finaliser
  k ^= k >> 30; k *= 0xbf58476d1ce4e5b9ull; k ^= k >> 27; k *= 0x94d049bb133111ebull; k ^= k >> 31;
  return k;
}
__device__ __forceinline__ long long vox_floor_div(double x, double v) { return (long long)floor(__ddiv_rn(x, v)); }

// Probe sequences are cut at kVoxMaxProbe slots: a key that finds neither itself nor an empty slot within that window is
// counted in `overflow` (the table is too full for it).  vox_contains walks the same window, so a stored key is always
// found.  At the load factors the sets are sized for (<= 0.5) linear probing essentially never reaches 128; an undersized
// table now costs at most 128 reads per key instead of `capacity`.
constexpr unsigned long long kVoxMaxProbe = 128;

__device__ __forceinline__ bool vox_insert(unsigned long long* table, unsigned long long mask, unsigned long long key,
                                           uint32_t* overflow) {
  unsigned long long slot = vox_hash(key) & mask;
  for (unsigned long long probe = 0; probe <= mask && probe < kVoxMaxProbe; ++probe) {
    const unsigned long long cur = table[slot];   // most insertions are duplicates: read before the atomic
    if (cur == key) return true;
    if (cur == kVoxEmpty) {
      const unsigned long long old = atomicCAS(table + slot, kVoxEmpty, key);
      if (old == kVoxEmpty || old == key) return true;
    }
    slot = (slot + 1) & mask;
  }
  atomicAdd(overflow, 1u);  // no room within the probe window
  return false;
}

__device__ __forceinline__ bool vox_contains(const unsigned long long* table, unsigned long long mask, unsigned long long key) {
  unsigned long long slot = vox_hash(key) & mask;
  for (unsigned long long probe = 0; probe <= mask && probe < kVoxMaxProbe; ++probe) {
    const unsigned long long cur = __ldg(table + slot);
    if (cur == key) return true;
    if (cur == kVoxEmpty) return false;
    slot = (slot + 1) & mask;
  }
  return false;
}

__global__ void __launch_bounds__(256) vox_clear_kernel(unsigned long long* table, int64_t cap) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < cap; i += stride) table[i] = kVoxEmpty;
}

// Eq. 20: every voxel meeting the closed axis-aligned box [mu - k s, mu + k s].  One thread per Gaussian; a box of up to
// kBoxInline voxels is inserted by its own thread, a larger one by the whole warp (lanes stride over the linearised box),
// so that one background Gaussian costs count / 32 inserts per lane instead of `count` in a single thread.  A box of more
// than kBoxMaxVoxels voxels is not inserted at all and counted in `overflow` (no table a caller would pass holds it).  On
// the warp path a lane stops at its first key that finds no room: the set is inexact from there on anyway (gs.h), and a
// full table then costs one failed probe window per lane and box instead of one per voxel.
constexpr unsigned long long kBoxInline = 64;
constexpr unsigned long long kBoxMaxVoxels = 1ull << 24;

__global__ void __launch_bounds__(128)
vox_boxes_kernel(unsigned long long* table, unsigned long long mask, double v, double k, int64_t N,
                 const float* __restrict__ means, const float* __restrict__ scales, uint32_t* overflow) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  long long lo[3] = {0, 0, 0};
  unsigned long long n[3] = {0, 0, 0}, count = 0;
  if (i < N) {
    long long hi[3];
    bool ok = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const double mu = (double)means[3 * i + a], h = __dmul_rn(k, (double)scales[3 * i + a]);
      ok = ok && isfinite(mu) && isfinite(h);        // floor(NaN) converts to 0: caught here, not by the range test
      lo[a] = vox_floor_div(__dsub_rn(mu, h), v);
      hi[a] = vox_floor_div(__dadd_rn(mu, h), v);
      ok = ok && vox_in_range(lo[a]) && vox_in_range(hi[a]) && hi[a] >= lo[a];
      n[a] = ok ? (unsigned long long)(hi[a] - lo[a] + 1) : 0ull;
    }
    count = n[0] * n[1] * n[2];                      // each factor <= 2^21
    if (!ok || count > kBoxMaxVoxels) { atomicAdd(overflow, 1u); count = 0; }
    if (count <= kBoxInline) {
      for (unsigned long long j = 0; j < count; ++j) {
        const unsigned long long ix = j % n[0], r = j / n[0];
        vox_insert(table, mask, vox_key(lo[0] + (long long)ix, lo[1] + (long long)(r % n[1]), lo[2] + (long long)(r / n[1])), overflow);
      }
      count = 0;
    }
  }
  // boxes left over: one at a time, spread over the warp
  const unsigned lane = threadIdx.x & 31;
  unsigned pending = __ballot_sync(0xffffffffu, count != 0);
  while (pending) {
    const int src = __ffs(pending) - 1;
    pending &= pending - 1;
    const long long l0 = __shfl_sync(0xffffffffu, lo[0], src), l1 = __shfl_sync(0xffffffffu, lo[1], src),
                    l2 = __shfl_sync(0xffffffffu, lo[2], src);
    const uint32_t n0 = (uint32_t)__shfl_sync(0xffffffffu, n[0], src), n1 = (uint32_t)__shfl_sync(0xffffffffu, n[1], src);
    const uint32_t cnt = (uint32_t)__shfl_sync(0xffffffffu, count, src);   // <= 2^24
    for (uint32_t j = lane; j < cnt; j += 32) {
      const uint32_t ix = j % n0, r = j / n0;
      if (!vox_insert(table, mask, vox_key(l0 + ix, l1 + (r % n1), l2 + (r / n1)), overflow)) break;
    }
  }
}

struct RayCam { double fx, fy, cx, cy, R[9], t[3]; int W, H, stride; };

// Eq. 21: 3-D DDA along c + t (r - c), t in [0, 1), one thread per (sub-sampled) pixel with depth > 0
__global__ void __launch_bounds__(128)
vox_rays_kernel(unsigned long long* table, unsigned long long mask, double v, RayCam cam, const float* __restrict__ depth,
                uint32_t* overflow) {
  const int nx = (cam.W + cam.stride - 1) / cam.stride, ny = (cam.H + cam.stride - 1) / cam.stride;
  const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= (int64_t)nx * ny) return;
  const int X = (int)(q % nx) * cam.stride, Y = (int)(q / nx) * cam.stride;
  const double z = (double)depth[(size_t)Y * cam.W + X];
  if (!(z > 0.0)) return;
  // camera centre c = -R^T t and surface point r = R^T (p_c - t), sums left to right, one rounding per operation
  double pc[3] = {__ddiv_rn(__dmul_rn(__dsub_rn((double)X, cam.cx), z), cam.fx),
                  __ddiv_rn(__dmul_rn(__dsub_rn((double)Y, cam.cy), z), cam.fy), z};
  double c[3], d[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    c[a] = -__dadd_rn(__dadd_rn(__dmul_rn(cam.R[a], cam.t[0]), __dmul_rn(cam.R[3 + a], cam.t[1])), __dmul_rn(cam.R[6 + a], cam.t[2]));
    const double q0 = __dsub_rn(pc[0], cam.t[0]), q1 = __dsub_rn(pc[1], cam.t[1]), q2 = __dsub_rn(pc[2], cam.t[2]);
    const double r = __dadd_rn(__dadd_rn(__dmul_rn(cam.R[a], q0), __dmul_rn(cam.R[3 + a], q1)), __dmul_rn(cam.R[6 + a], q2));
    d[a] = __dsub_rn(r, c[a]);
  }
  long long idx[3], step[3];
  double t_max[3], t_delta[3];
  bool ok = true;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    idx[a] = vox_floor_div(c[a], v);
    ok = ok && vox_in_range(idx[a]) && isfinite(d[a]);
    step[a] = 0; t_max[a] = INFINITY; t_delta[a] = INFINITY;
    if (d[a] > 0.0) {
      step[a] = 1;
      t_max[a] = __ddiv_rn(__dsub_rn(__dmul_rn(__dadd_rn((double)idx[a], 1.0), v), c[a]), d[a]);
      t_delta[a] = __ddiv_rn(v, d[a]);
    } else if (d[a] < 0.0) {
      step[a] = -1;
      t_max[a] = __ddiv_rn(__dsub_rn(__dmul_rn((double)idx[a], v), c[a]), d[a]);
      t_delta[a] = __ddiv_rn(-v, d[a]);
    }
  }
  if (!ok) { atomicAdd(overflow, 1u); return; }
  if (!vox_insert(table, mask, vox_key(idx[0], idx[1], idx[2]), overflow)) return;   // table full: give the ray up
  for (int guard = 0; guard < (1 << 22); ++guard) {
    int a = 0;                                   // axis of the nearest boundary; ties -> lowest axis
    if (t_max[1] < t_max[a]) a = 1;
    if (t_max[2] < t_max[a]) a = 2;
    const double tm = a == 0 ? t_max[0] : (a == 1 ? t_max[1] : t_max[2]);
    if (!(tm < 1.0)) break;                      // the next boundary lies at t >= 1
    if (a == 0) { idx[0] += step[0]; t_max[0] = __dadd_rn(t_max[0], t_delta[0]); }
    else if (a == 1) { idx[1] += step[1]; t_max[1] = __dadd_rn(t_max[1], t_delta[1]); }
    else { idx[2] += step[2]; t_max[2] = __dadd_rn(t_max[2], t_delta[2]); }
    if (!(vox_in_range(idx[0]) && vox_in_range(idx[1]) && vox_in_range(idx[2]))) { atomicAdd(overflow, 1u); return; }
    if (!vox_insert(table, mask, vox_key(idx[0], idx[1], idx[2]), overflow)) return;
  }
}

// Eq. 22: retained iff kappa(mu) is in neither set
__global__ void __launch_bounds__(256)
vox_retain_kernel(const unsigned long long* occ, unsigned long long occ_mask, const unsigned long long* fre,
                  unsigned long long free_mask, double v, int64_t N, const float* __restrict__ means, uint8_t* __restrict__ retain) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const float m0 = means[3 * i], m1 = means[3 * i + 1], m2 = means[3 * i + 2];
  const long long ix = vox_floor_div((double)m0, v), iy = vox_floor_div((double)m1, v), iz = vox_floor_div((double)m2, v);
  bool keep = isfinite(m0) && isfinite(m1) && isfinite(m2);   // a Gaussian without a position is never retained (gs.h)
  if (keep && vox_in_range(ix) && vox_in_range(iy) && vox_in_range(iz)) {
    const unsigned long long key = vox_key(ix, iy, iz);
    if (occ && vox_contains(occ, occ_mask, key)) keep = false;
    if (keep && fre && vox_contains(fre, free_mask, key)) keep = false;
  }
  retain[i] = keep ? 1 : 0;
}

static bool pow2(int64_t c) { return c >= 2 && (c & (c - 1)) == 0; }

}  // namespace gs

using namespace gs;

extern "C" {

int gs_voxel_set_clear(void* stream, uint64_t* table, int64_t capacity) {
  if (!table || !pow2(capacity)) return GS_E_INVALID;
  int64_t g = div_up(capacity, 256);
  if (g > 148 * 16) g = 148 * 16;
  vox_clear_kernel<<<(int)g, 256, 0, (cudaStream_t)stream>>>(reinterpret_cast<unsigned long long*>(table), capacity);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

int gs_voxel_insert_boxes(void* stream, uint64_t* table, int64_t capacity, float voxel, float k, int64_t N,
                          const float* means, const float* scales, uint32_t* overflow) {
  if (!table || !pow2(capacity) || !(voxel > 0.f) || !isfinite(voxel) || !(k >= 0.f) || !isfinite(k) || N < 0 || !overflow || (N > 0 && (!means || !scales)))
    return GS_E_INVALID;
  if (N == 0) return GS_OK;
  vox_boxes_kernel<<<(unsigned)div_up(N, 128), 128, 0, (cudaStream_t)stream>>>(
      reinterpret_cast<unsigned long long*>(table), (unsigned long long)capacity - 1ull, (double)voxel, (double)k, N, means,
      scales, overflow);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

int gs_voxel_insert_rays(void* stream, uint64_t* table, int64_t capacity, float voxel, const gs_camera* cam,
                         const float* depth, int32_t stride, uint32_t* overflow) {
  if (!table || !pow2(capacity) || !(voxel > 0.f) || !isfinite(voxel) || !cam || !depth || stride < 1 || !overflow || cam->width <= 0 ||
      cam->height <= 0)
    return GS_E_INVALID;
  RayCam rc;
  rc.fx = cam->fx; rc.fy = cam->fy; rc.cx = cam->cx; rc.cy = cam->cy;
  for (int r = 0; r < 3; ++r) {
    for (int c = 0; c < 3; ++c) rc.R[3 * r + c] = cam->T_cw[4 * r + c];
    rc.t[r] = cam->T_cw[4 * r + 3];
  }
  rc.W = cam->width; rc.H = cam->height; rc.stride = stride;
  const int64_t n = (int64_t)((cam->width + stride - 1) / stride) * ((cam->height + stride - 1) / stride);
  vox_rays_kernel<<<(unsigned)div_up(n, 128), 128, 0, (cudaStream_t)stream>>>(
      reinterpret_cast<unsigned long long*>(table), (unsigned long long)capacity - 1ull, (double)voxel, rc, depth, overflow);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

int gs_voxel_retain(void* stream, const uint64_t* occ, int64_t occ_capacity, const uint64_t* free_set, int64_t free_capacity,
                    float voxel, int64_t N, const float* means, uint8_t* retain) {
  if ((occ && !pow2(occ_capacity)) || (free_set && !pow2(free_capacity)) || !(voxel > 0.f) || !isfinite(voxel) || N < 0 ||
      (N > 0 && (!means || !retain)))
    return GS_E_INVALID;
  if (N == 0) return GS_OK;
  vox_retain_kernel<<<(unsigned)div_up(N, 256), 256, 0, (cudaStream_t)stream>>>(
      reinterpret_cast<const unsigned long long*>(occ), occ ? (unsigned long long)occ_capacity - 1ull : 0ull,
      reinterpret_cast<const unsigned long long*>(free_set), free_set ? (unsigned long long)free_capacity - 1ull : 0ull,
      (double)voxel, N, means, retain);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

}  // extern "C"

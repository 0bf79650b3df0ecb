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

// gs_normals.cu -- depth-induced normals of the rendered depth map and the normal term of Eqs. 4 / 23 (PAPER.md:86:
// "L_normal = sum_k |1 - N^_k^T N-_k| ... between the depth-induced normal N^_k and the monocular normal prior N-_k"; rendered
// normals: PAPER.md:133, 393).  Reading Q22: p(u,v) = ((u - cx) D / fx, (v - cy) D / fy, D), forward differences
// t_x = p(u+1,v) - p(u,v), t_y = p(u,v+1) - p(u,v), N^ = (t_y x t_x) / |t_y x t_x|; a pixel has a normal iff it is not in the
// last column / row and its three depths are > 0; the prior is valid where non-zero; mean over all H W pixels.
// One thread per pixel.  The gradient w.r.t. the depth map is GATHERED: depth pixel (u,v) enters the normals of (u,v),
// (u-1,v) and (u,v-1), so every thread re-forms those three normals and adds their three contributions -- deterministic,
// no atomics.  HBM-bound: 4 + 12 B read (+ neighbours from L1/L2), 4 (+ 12) B written per pixel.
// Product code: nothing here includes, links or calls oracle/.
#include "gs_internal.cuh"

namespace gs {

struct NCam { float fx, fy, cx, cy; int W, H; };

struct V3 { float x, y, z; };
__device__ __forceinline__ V3 v3(float x, float y, float z) { V3 r = {x, y, z}; return r; }
__device__ __forceinline__ V3 sub(V3 a, V3 b) { return v3(a.x - b.x, a.y - b.y, a.z - b.z); }
__device__ __forceinline__ V3 cross(V3 a, V3 b) { return v3(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x); }
__device__ __forceinline__ float dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }

__device__ __forceinline__ V3 ray_of(const NCam& c, int x, int y) { return v3(((float)x - c.cx) / c.fx, ((float)y - c.cy) / c.fy, 1.f); }

// Normal of pixel (x, y) and, if `prior` is given, the gradients of |1 - n . prior| w.r.t. the three depths it uses.
// Returns false if the pixel has no normal.  g0, gx, gy: dL/dD(x,y), dL/dD(x+1,y), dL/dD(x,y+1) (unscaled).
__device__ __forceinline__ bool normal_terms(const NCam& c, const float* __restrict__ depth, const float* __restrict__ prior,
                                             int x, int y, V3& n, float& e, float& g0, float& gx, float& gy) {
  if (x < 0 || y < 0 || x + 1 >= c.W || y + 1 >= c.H) return false;
  const float d0 = depth[(size_t)y * c.W + x], dx = depth[(size_t)y * c.W + x + 1], dy = depth[(size_t)(y + 1) * c.W + x];
  if (!(d0 > 0.f && dx > 0.f && dy > 0.f)) return false;
  const V3 r0 = ray_of(c, x, y), rx = ray_of(c, x + 1, y), ry = ray_of(c, x, y + 1);
  // t_x = p(x+1,y) - p(x,y) = ray(x,y) (dx - d0) + (dx / fx, 0, 0): written with the depth DIFFERENCE (exact in fp32 for
  // nearby depths) so that the tangents do not cancel two numbers of the size of the point coordinates
  const float ex = dx - d0, ey = dy - d0;
  const V3 tx = v3(fmaf(r0.x, ex, dx / c.fx), r0.y * ex, ex), ty = v3(r0.x * ey, fmaf(r0.y, ey, dy / c.fy), ey);
  const V3 cr = cross(ty, tx);
  const float l2 = dot(cr, cr);
  if (!(l2 > 0.f)) return false;
  const float il = rsqrtf(l2);
  n = v3(cr.x * il, cr.y * il, cr.z * il);
  e = 0.f; g0 = gx = gy = 0.f;
  if (prior) {
    const size_t HW = (size_t)c.W * c.H, p = (size_t)y * c.W + x;
    const V3 nb = v3(prior[p], prior[HW + p], prior[2 * HW + p]);
    if (nb.x == 0.f && nb.y == 0.f && nb.z == 0.f) return true;   // no prior here: a normal, but no loss
    e = 1.f - dot(n, nb);
    const float sg = e > 0.f ? -1.f : (e < 0.f ? 1.f : 0.f);       // dL/dn = -sign(e) nb
    const V3 gn = v3(sg * nb.x, sg * nb.y, sg * nb.z);
    const float ng = dot(n, gn);
    const V3 gc = v3((gn.x - n.x * ng) * il, (gn.y - n.y * ng) * il, (gn.z - n.z * ng) * il);
    const V3 gty = cross(tx, gc), gtx = cross(gc, ty);
    gx = dot(rx, gtx);
    gy = dot(ry, gty);
    g0 = -dot(r0, v3(gtx.x + gty.x, gtx.y + gty.y, gtx.z + gty.z));
  }
  return true;
}

__global__ void __launch_bounds__(256)
normal_kernel(NCam c, const float* __restrict__ depth, const float* __restrict__ prior, float weight,
              float* __restrict__ normals_out, float* __restrict__ d_depth, double* __restrict__ sums) {
  const int x = blockIdx.x * 32 + (threadIdx.x & 31), y = blockIdx.y * 8 + (threadIdx.x >> 5);
  double acc = 0.0;
  if (x < c.W && y < c.H) {
    const size_t HW = (size_t)c.W * c.H, p = (size_t)y * c.W + x;
    V3 n = v3(0.f, 0.f, 0.f), m;
    float e, g0, gx, gy, g = 0.f;
    const bool has = normal_terms(c, depth, prior, x, y, n, e, g0, gx, gy);
    if (has) { acc = (double)fabsf(e); g += g0; } else n = v3(0.f, 0.f, 0.f);
    if (normals_out) { normals_out[p] = n.x; normals_out[HW + p] = n.y; normals_out[2 * HW + p] = n.z; }
    if (prior && d_depth) {
      if (normal_terms(c, depth, prior, x - 1, y, m, e, g0, gx, gy)) g += gx;   // this pixel is the x+1 neighbour of (x-1, y)
      if (normal_terms(c, depth, prior, x, y - 1, m, e, g0, gx, gy)) g += gy;   // ... and the y+1 neighbour of (x, y-1)
      d_depth[p] += weight * g;
    }
  }
  // block sum of the loss terms
  __shared__ double s_a[8];
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
  if ((threadIdx.x & 31) == 0) s_a[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0 && sums) {
    double t = 0.0;
    for (int w = 0; w < 8; ++w) t += s_a[w];
    if (t != 0.0) atomicAdd(sums + 1, t);
  }
}

__global__ void normal_final_kernel(double* sums, double inv_p, double lambda_n) {
  if (threadIdx.x == 0 && blockIdx.x == 0) sums[0] = lambda_n * sums[1] * inv_p;
}

}  // namespace gs

using namespace gs;

extern "C" int gs_loss_normal(void* stream, int32_t width, int32_t height, float fx, float fy, float cx, float cy,
                              const float* depth, const float* normal_prior, float lambda_n, float* normals_out,
                              float* d_depth, double* loss) {
  if (width <= 0 || height <= 0 || !depth || !(fx > 0.f) || !(fy > 0.f)) return GS_E_INVALID;
  if (normal_prior && (!d_depth || !loss)) return GS_E_INVALID;
  if (!normal_prior && !normals_out) return GS_E_INVALID;
  cudaStream_t s = (cudaStream_t)stream;
  if (loss && cudaMemsetAsync(loss, 0, 2 * sizeof(double), s) != cudaSuccess) { cudaGetLastError(); return GS_E_CUDA; }
  const NCam c = {fx, fy, cx, cy, width, height};
  const double inv_p = 1.0 / ((double)width * height);
  const dim3 grid((width + 31) / 32, (height + 7) / 8);
  normal_kernel<<<grid, 256, 0, s>>>(c, depth, normal_prior, (float)((double)lambda_n * inv_p), normals_out,
                                     normal_prior ? d_depth : nullptr, normal_prior ? loss : nullptr);
  if (normal_prior) normal_final_kernel<<<1, 32, 0, s>>>(loss, inv_p, (double)lambda_n);
  return cudaGetLastError() == cudaSuccess ? GS_OK : GS_E_CUDA;
}

// gs_preprocess.cu -- step a1: per-Gaussian EWA projection, conic, screen extent, SH colour.
// HBM-bound: reads 44 B per Gaussian (+12K B of SH if visible), writes ~120 B per visible Gaussian.
#include "gs_internal.cuh"
#include "gs_project.cuh"
#include "gs_raster.cuh"
#include "gs_sh.cuh"

#ifndef GS_PRE_CTAS_PER_SM
#define GS_PRE_CTAS_PER_SM 4
#endif

namespace gs {

// Persistent CTAs of 128 threads.  Two phases (evidence: profiles/r2_stages.md -- with one thread per Gaussian doing
// everything, the third of the Gaussians that is visible was spread evenly over every warp: the fp64 projection chain, the
// SH evaluation and the record writes ran at 18 of 32 lanes, and every thread walked its own 192-byte SH row):
//   CULL   U (1, 2 or 4) Gaussians per thread and round, all their loads in flight at once: a cheap fp32 test that can only err on the side of keeping (behind the
//          near plane with a rounding margin; opacity < 1/255, exact; a bound of the footprint -- rho sqrt(s_max^2 |J|_F^2
//          + 0.3), which dominates both half widths of the exact extent -- that misses the image).  Survivors are appended
//          to a queue in shared memory; the rest get tiles_touched = 0 and are done.
//   HEAVY  whenever the queue holds 128 candidates (and once at the end for the rest): one thread per candidate runs the
//          fp64 chain, the exact cull and the tile rect exactly as before -- the decisions cannot differ -- while the SH rows
//          of the 128 candidates arrive in shared memory through cp.async issued by the whole CTA (consecutive lanes fetch
//          consecutive 16 bytes of a row); the colour is then evaluated from the thread's row (row stride 52 floats:
//          conflict-free LDS.128).
constexpr int kPreT = 128;
constexpr int kPreUMax = 4;  // Gaussians per thread and round of the cull phase (template parameter U: 1, 2 or 4)

template <int DEG, int kPreU>
__global__ void __launch_bounds__(kPreT, GS_PRE_CTAS_PER_SM)
preprocess_kernel(int64_t N, const float* __restrict__ means, const float* __restrict__ scales,
                  const float* __restrict__ quats, const float* __restrict__ opacities, const float* __restrict__ sh,
                  DevCam cam, float4* __restrict__ feat,
                  uint32_t* __restrict__ tiles_touched, uint32_t* __restrict__ tile_count,
                  uint32_t* __restrict__ vis_ids, uint4* __restrict__ vis_rec, float4* __restrict__ vis_par,
                  uint32_t* __restrict__ slot_of, Counts* __restrict__ counts, double* __restrict__ pose_acc) {
  constexpr int K = (DEG + 1) * (DEG + 1);
  constexpr int K3 = 3 * K;
  constexpr bool V4 = (K3 % 4) == 0;
  constexpr int RS = V4 ? ((K3 / 4) % 2 ? K3 : K3 + 4) : K3;  // row stride in floats (gs_gauss_bwd.cu uses the same layout)
  constexpr int EW = V4 ? 4 : 1, EPR = K3 / EW;
  __shared__ __align__(16) float s_sh[kPreT * RS];
  __shared__ uint32_t s_q[(kPreUMax + 1) * kPreT];  // candidate queue (Gaussian indices)
  __shared__ uint32_t s_wcnt[kPreT / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  pdl_enter();
  if (blockIdx.x == 0 && tid < 16) pose_acc[tid] = 0.0;  // accumulated by gauss_bwd_kernel of this iteration
  float T[12];
  load_pose(cam, T);
  // view direction mu - c_cam, c_cam = -W^T t
  const double ccx = -((double)T[0] * T[3] + (double)T[4] * T[7] + (double)T[8] * T[11]);
  const double ccy = -((double)T[1] * T[3] + (double)T[5] * T[7] + (double)T[9] * T[11]);
  const double ccz = -((double)T[2] * T[3] + (double)T[6] * T[7] + (double)T[10] * T[11]);
  const float fW = (float)cam.W, fH = (float)cam.H;
  const float f2sum = cam.fx * cam.fx + cam.fy * cam.fy;

  // HEAVY phase for the first nb (<= 128) candidates of the queue
  auto heavy = [&](int h0, int nb) {
    for (int f = tid; f < nb * EPR; f += kPreT) {
      const int r = f / EPR, c = f - r * EPR;
      const float* src = sh + (int64_t)K3 * s_q[h0 + r] + c * EW;
      if constexpr (V4) cp_async16(s_sh + r * RS + c * EW, src); else cp_async4(s_sh + r * RS + c * EW, src);
    }
    bool vis = false;
    int64_t i = 0;
    float mu0 = 0.f, mu1 = 0.f, mu2 = 0.f, o = 0.f, sc0 = 0.f, sc1 = 0.f, sc2 = 0.f;
    float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
    ProjD P;
    int tx0 = 0, ty0 = 0, tx1 = 0, ty1 = 0;
    if (tid < nb) {
      i = (int64_t)s_q[h0 + tid];
      mu0 = means[3 * i]; mu1 = means[3 * i + 1]; mu2 = means[3 * i + 2];
      sc0 = scales[3 * i]; sc1 = scales[3 * i + 1]; sc2 = scales[3 * i + 2];
      o = opacities[i];
      q = *reinterpret_cast<const float4*>(quats + 4 * i);
      vis = project_gaussian<double>(cam, T, mu0, mu1, mu2, sc0, sc1, sc2, q.x, q.y, q.z, q.w, o, P);
      if (vis) vis = tile_rect(cam, P, o, tx0, ty0, tx1, ty1);
      tiles_touched[i] = vis ? (uint32_t)((tx1 - tx0) * (ty1 - ty0)) : 0u;
    }
    // Compacted list of visible Gaussians (arbitrary order).  Everything downstream is indexed by the visible slot: the
    // feature records, the parameter copies and the 2-D gradient accumulators of the visible Gaussians are dense
    // arrays -- sequential streams for the per-Gaussian kernels and a third of the footprint for the gathers of the
    // compositing kernels.
    const unsigned ball = __ballot_sync(0xffffffffu, vis);
    uint32_t base = 0;
    if (lane == 0 && ball) base = atomicAdd(&counts->n_visible, (uint32_t)__popc(ball));
    base = __shfl_sync(0xffffffffu, base, 0);
    const size_t slot = base + __popc(ball & ((1u << lane) - 1));
    cp_async_wait_all();
    __syncthreads();  // the SH rows of the batch have landed
    if (vis) {
      const double vx = (double)mu0 - ccx, vy = (double)mu1 - ccy, vz = (double)mu2 - ccz;
      const float ivn = rsqrtf((float)(vx * vx + vy * vy + vz * vz));
      float B[K];
      sh_basis<DEG>((float)vx * ivn, (float)vy * ivn, (float)vz * ivn, B);
      const float* row = s_sh + tid * RS;
      float col[3] = {0.f, 0.f, 0.f};
      if constexpr (V4) {
#pragma unroll
        for (int v = 0; v < K3 / 4; ++v) {
          const float4 t = *reinterpret_cast<const float4*>(row + 4 * v);
          const float e[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
          for (int u = 0; u < 4; ++u) col[(4 * v + u) % 3] = fmaf(B[(4 * v + u) / 3], e[u], col[(4 * v + u) % 3]);
        }
      } else {
#pragma unroll
        for (int k = 0; k < K3; ++k) col[k % 3] = fmaf(B[k / 3], row[k], col[k % 3]);
      }
      // mean = integer pixel (two int16, clamped: a centre that far off-screen needs no sub-pixel precision) + fraction
      const double rmx = fmin(fmax(rint(P.mx), -32000.0), 32000.0);
      const double rmy = fmin(fmax(rint(P.my), -32000.0), 32000.0);
      // whitened conic (gs_raster.cuh): 0.5 log2(e) d^T Q d = u^2 + v^2, u = l11 dx + l21 dy, v = l22 dy; fp64 Cholesky,
      // k c - l21^2 = k det(Q) / a > 0 for the positive-definite Q that passed the cull
      const double kh = 0.5 * 1.4426950408889634;  // 0.5 log2(e)
      const double l11 = sqrt(kh * P.a), l21 = kh * P.b / l11, l22 = sqrt(kh * (P.c - P.b * P.b / P.a));
      float4 f0, f1, f2;
      f0.x = (float)(P.mx - rmx); f0.y = (float)(P.my - rmy);
      f0.z = __int_as_float(((int)rmy << 16) | ((int)rmx & 0xffff));
      f0.w = o;
      f1.x = (float)l11; f1.y = (float)l21; f1.z = (float)l22; f1.w = (float)log2((double)o);
      f2.x = fmaxf(col[0] + 0.5f, 0.f); f2.y = fmaxf(col[1] + 0.5f, 0.f); f2.z = fmaxf(col[2] + 0.5f, 0.f);
      f2.w = (float)P.z;
      const uint32_t dk = __float_as_uint(depth_key_f32(T, mu0, mu1, mu2));
      vis_ids[slot] = (uint32_t)i;
      slot_of[i] = (uint32_t)slot;
      // what the duplication needs: packed tile rect, depth key, index
      vis_rec[slot] = make_uint4((uint32_t)tx0 | ((uint32_t)ty0 << 16), (uint32_t)tx1 | ((uint32_t)ty1 << 16), dk, (uint32_t)i);
      feat[3 * slot] = f0; feat[3 * slot + 1] = f1; feat[3 * slot + 2] = f2;
      // the parameters the per-Gaussian backward needs again
      vis_par[3 * slot] = make_float4(mu0, mu1, mu2, o);
      vis_par[3 * slot + 1] = make_float4(sc0, sc1, sc2, 0.f);
      vis_par[3 * slot + 2] = q;
      for (int ty = ty0; ty < ty1; ++ty)  // MSD digit histogram of the binning sort (gs_binning.cu)
        for (int tx = tx0; tx < tx1; ++tx) atomicAdd(&tile_count[(size_t)(ty * cam.tiles_x + tx) * kCtrStride], 1u);
    }
    __syncthreads();  // s_sh is free again
  };

  // CULL phase: kPreU Gaussians per thread and round, all their loads in flight before the first test (the kernel is a
  // chain of DRAM round trips: what counts is how many bytes each SM has outstanding)
  int qn = 0, head = 0;  // candidates in the queue / start of the queue (uniform over the CTA)
  const int64_t nchunks = (N + kPreT * kPreU - 1) / (kPreT * kPreU);
  for (int64_t chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x) {
    float m0[kPreU], m1[kPreU], m2[kPreU], op[kPreU], s0[kPreU], s1[kPreU], s2[kPreU];
#pragma unroll
    for (int u = 0; u < kPreU; ++u) {
      const int64_t i = (chunk * kPreU + u) * kPreT + tid;
      const bool in = i < N;
      m0[u] = in ? means[3 * i] : 0.f; m1[u] = in ? means[3 * i + 1] : 0.f; m2[u] = in ? means[3 * i + 2] : 0.f;
      s0[u] = in ? scales[3 * i] : 0.f; s1[u] = in ? scales[3 * i + 1] : 0.f; s2[u] = in ? scales[3 * i + 2] : 0.f;
      op[u] = in ? opacities[i] : 0.f;
    }
    bool cand[kPreU];
#pragma unroll
    for (int u = 0; u < kPreU; ++u) {
      const int64_t i = (chunk * kPreU + u) * kPreT + tid;
      const float mu0 = m0[u], mu1 = m1[u], mu2 = m2[u], o = op[u];
      const float smax = fmaxf(s0[u], fmaxf(s1[u], s2[u]));
      const float zc = depth_key_f32(T, mu0, mu1, mu2);
      const float xc = fmaf(T[0], mu0, fmaf(T[1], mu1, fmaf(T[2], mu2, T[3]))), yc = fmaf(T[4], mu0, fmaf(T[5], mu1, fmaf(T[6], mu2, T[7])));
      // rounding margin of the fp32 depth against the fp64 one the exact test uses
      const float az = fabsf(T[8] * mu0) + fabsf(T[9] * mu1) + fabsf(T[10] * mu2) + fabsf(T[11]);
      const bool behind = zc < cam.near_z - 4e-6f * az;
      const bool faint = (double)o < 1.0 / 255.0;
      const float iz = 1.f / zc, mx = cam.fx * xc * iz + cam.cx, my = cam.fy * yc * iz + cam.cy;
      const float jf2 = (f2sum + (cam.fx * cam.fx * xc * xc + cam.fy * cam.fy * yc * yc) * iz * iz) * iz * iz;  // |J|_F^2
      const float rho2 = 2.f * __logf(255.f * o) * 1.001f + 1e-3f;
      const float bnd = sqrtf(rho2 * fmaf(smax * smax, jf2, GS_DILATION)) * 1.01f + 1.f + 1e-3f * (fabsf(mx) + fabsf(my));
      // "provably outside": every comparison is false for a NaN, which therefore stays a candidate
      const bool outside = (mx + bnd < 0.f) || (mx - bnd > fW) || (my + bnd < 0.f) || (my - bnd > fH);
      cand[u] = i < N && !behind && !faint && !outside;
      if (i < N && !cand[u]) tiles_touched[i] = 0u;
      if (cand[u] && K3 >= 12) {  // start the SH row on its way to L2
        const char* row = reinterpret_cast<const char*>(sh + (int64_t)K3 * i);
#pragma unroll
        for (int b = 0; b < 4 * K3; b += 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(row + b));
      }
    }
    // append the candidates to the queue (any order): rank inside the warp (ballots) + warp offsets (shared memory)
    unsigned bal[kPreU];
    int mine = 0;
#pragma unroll
    for (int u = 0; u < kPreU; ++u) { bal[u] = __ballot_sync(0xffffffffu, cand[u]); mine += __popc(bal[u]); }
    if (lane == 0) s_wcnt[warp] = mine;
    __syncthreads();
    int before = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kPreT / 32; ++w) { const int c = (int)s_wcnt[w]; before += w < warp ? c : 0; total += c; }
    int pos = head + qn + before;
#pragma unroll
    for (int u = 0; u < kPreU; ++u) {
      if (cand[u]) s_q[pos + __popc(bal[u] & ((1u << lane) - 1u))] = (uint32_t)((chunk * kPreU + u) * kPreT + tid);
      pos += __popc(bal[u]);
    }
    qn += total;
    __syncthreads();
    while (qn >= kPreT) { heavy(head, kPreT); head += kPreT; qn -= kPreT; }
    if (head > 0) {  // move the rest (< 128 entries) to the front
      const uint32_t moved = tid < qn ? s_q[head + tid] : 0u;
      __syncthreads();
      if (tid < qn) s_q[tid] = moved;
      head = 0;
      __syncthreads();
    }
  }
  if (qn > 0) heavy(head, qn);
}

int launch_preprocess(gs_ctx* ctx, cudaStream_t s) {
  const int64_t N = ctx->N;
  if (N == 0) return GS_OK;
  const int threads = kPreT;
  int sms = 148;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->device);
  // Gaussians per thread and round of the cull phase: 4 when that still gives every resident CTA a round (measured on
  // config 3: 1 / 2 / 4 / 8 -> 29.3 / 29.0 / 27.5 / 36.2 us), fewer for small scenes (config 2: 50 k Gaussians)
  const int64_t resident = (int64_t)sms * GS_PRE_CTAS_PER_SM;
  const int U = N >= 3 * resident * threads ? 4 : (N >= 2 * resident * threads ? 2 : 1);
  const unsigned blocks = (unsigned)min(resident, div_up(N, threads * U));  // persistent CTAs
#define GS_PRE_U(D, UU)                                                                                              \
  GS_LAUNCH_PDL((preprocess_kernel<D, UU>), blocks, threads, 0, s, N, ctx->means, ctx->scales, ctx->quats, ctx->opacities, \
                ctx->sh, ctx->cam, ctx->feat, ctx->tiles_touched, ctx->tile_count, ctx->vis_ids, ctx->vis_rec,        \
                ctx->vis_par, ctx->slot_of, ctx->counts, ctx->pose_acc)
#define GS_PRE(D)                                                                                                    \
  do {                                                                                                               \
    if (U == 4) GS_PRE_U(D, 4); else if (U == 2) GS_PRE_U(D, 2); else GS_PRE_U(D, 1);                                \
  } while (0)
  switch (ctx->sh_degree) {
    case 0: GS_PRE(0); break;
    case 1: GS_PRE(1); break;
    case 2: GS_PRE(2); break;
    default: GS_PRE(3); break;
  }
#undef GS_PRE
#undef GS_PRE_U
  GS_LAUNCH_CHECK("preprocess_kernel");
  return GS_OK;
}

}  // namespace gs

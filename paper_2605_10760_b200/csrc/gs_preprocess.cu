// gs_preprocess.cu -- step a1: per-Gaussian EWA projection, conic, screen extent, SH colour.
// One thread per Gaussian; HBM-bound: reads 44 B (+12K B of SH if visible), writes 64 B per visible Gaussian.
#include "gs_internal.cuh"
#include "gs_project.cuh"
#include "gs_sh.cuh"

namespace gs {

template <int DEG>
__global__ void __launch_bounds__(128, 8)
preprocess_kernel(int64_t N, const float* __restrict__ means, const float* __restrict__ scales,
                  const float* __restrict__ quats, const float* __restrict__ opacities, const float* __restrict__ sh,
                  DevCam cam, float4* __restrict__ feat,
                  uint32_t* __restrict__ tiles_touched, uint32_t* __restrict__ tile_count,
                  uint32_t* __restrict__ vis_ids, uint4* __restrict__ vis_rec, float4* __restrict__ vis_par,
                  uint32_t* __restrict__ slot_of, Counts* __restrict__ counts, double* __restrict__ pose_acc) {
  constexpr int K = (DEG + 1) * (DEG + 1);
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  pdl_enter();
  if (blockIdx.x == 0 && threadIdx.x < 16) pose_acc[threadIdx.x] = 0.0;  // accumulated by gauss_bwd_kernel of this iteration
  float T[12];
  load_pose(cam, T);
  bool vis = false;
  float mu0 = 0.f, mu1 = 0.f, mu2 = 0.f, o = 0.f, sc0 = 0.f, sc1 = 0.f, sc2 = 0.f;
  float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
  ProjD P;
  int tx0 = 0, ty0 = 0, tx1 = 0, ty1 = 0;
  if (i < N) {
    mu0 = means[3 * i]; mu1 = means[3 * i + 1]; mu2 = means[3 * i + 2];
    sc0 = scales[3 * i]; sc1 = scales[3 * i + 1]; sc2 = scales[3 * i + 2];
    o = opacities[i];
    q = *reinterpret_cast<const float4*>(quats + 4 * i);
    {
      // The SH row (12 K bytes) is only read if the Gaussian turns out visible, i.e. after the whole fp64 chain: a cheap
      // fp32 guess (in front of the near plane, centre within the image grown by ~4 sigma_max) starts it on its way to L2
      // now (measured A/B on one box: preprocess 32.3 -> 31.9 us; the same prefetch in gauss_bwd cost +1.7 us and a
      // warp-cooperative tile-count loop gained nothing here and cost emit_kernel 4 us: both reverted, profiles/r2_stages.md).
      const float zc = depth_key_f32(T, mu0, mu1, mu2);
      const float xc = fmaf(T[0], mu0, fmaf(T[1], mu1, fmaf(T[2], mu2, T[3]))), yc = fmaf(T[4], mu0, fmaf(T[5], mu1, fmaf(T[6], mu2, T[7])));
      const float iz = 1.f / fmaxf(zc, 1e-6f), m = 4.f * fmaxf(sc0, fmaxf(sc1, sc2)) * fmaxf(cam.fx, cam.fy) * iz + 8.f;
      const float u = cam.fx * xc * iz + cam.cx, v = cam.fy * yc * iz + cam.cy;
      if (zc > cam.near_z && u > -m && u < (float)cam.W + m && v > -m && v < (float)cam.H + m) {
        const char* row = reinterpret_cast<const char*>(sh + (int64_t)3 * K * i);
#pragma unroll
        for (int b = 0; b < 12 * K; b += 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(row + b));
      }
    }
    vis = project_gaussian<double>(cam, T, mu0, mu1, mu2, sc0, sc1, sc2, q.x, q.y, q.z, q.w, o, P);
    if (vis) vis = tile_rect(cam, P, o, tx0, ty0, tx1, ty1);
    tiles_touched[i] = vis ? (uint32_t)((tx1 - tx0) * (ty1 - ty0)) : 0u;
  }
  // Compacted list of visible Gaussians (arbitrary order).  Everything downstream is indexed by the visible slot: the
  // feature records, the parameter copies and the 2-D gradient accumulators of the visible Gaussians are dense
  // arrays -- sequential streams for the per-Gaussian kernels (their scattered 64-byte DRAM bursts, ~9 per Gaussian,
  // were what bounded them) and a third of the footprint for the gathers of the compositing kernels.
  const unsigned ball = __ballot_sync(0xffffffffu, vis);
  if (ball == 0) return;
  const int lane = threadIdx.x & 31;
  uint32_t base = 0;
  if (lane == 0) base = atomicAdd(&counts->n_visible, (uint32_t)__popc(ball));
  base = __shfl_sync(0xffffffffu, base, 0);
  if (!vis) return;
  const size_t slot = base + __popc(ball & ((1u << lane) - 1));
  // view direction mu - c_cam, c_cam = -W^T t
  const double ccx = -((double)T[0] * T[3] + (double)T[4] * T[7] + (double)T[8] * T[11]);
  const double ccy = -((double)T[1] * T[3] + (double)T[5] * T[7] + (double)T[9] * T[11]);
  const double ccz = -((double)T[2] * T[3] + (double)T[6] * T[7] + (double)T[10] * T[11]);
  const double vx = (double)mu0 - ccx, vy = (double)mu1 - ccy, vz = (double)mu2 - ccz;
  const float ivn = rsqrtf((float)(vx * vx + vy * vy + vz * vz));
  float B[K];
  sh_basis<DEG>((float)vx * ivn, (float)vy * ivn, (float)vz * ivn, B);
  const float* c = sh + (int64_t)3 * K * i;
  float col[3] = {0.f, 0.f, 0.f};
  if constexpr ((3 * K) % 4 == 0) {
    float buf[3 * K];
#pragma unroll
    for (int v = 0; v < 3 * K / 4; ++v) {
      const float4 t = __ldg(reinterpret_cast<const float4*>(c) + v);
      buf[4 * v] = t.x; buf[4 * v + 1] = t.y; buf[4 * v + 2] = t.z; buf[4 * v + 3] = t.w;
    }
#pragma unroll
    for (int k = 0; k < K; ++k) {
      col[0] = fmaf(B[k], buf[3 * k], col[0]);
      col[1] = fmaf(B[k], buf[3 * k + 1], col[1]);
      col[2] = fmaf(B[k], buf[3 * k + 2], col[2]);
    }
  } else {
#pragma unroll
    for (int k = 0; k < K; ++k) {
      const float c0 = __ldg(c + 3 * k), c1 = __ldg(c + 3 * k + 1), c2 = __ldg(c + 3 * k + 2);
      col[0] = fmaf(B[k], c0, col[0]);
      col[1] = fmaf(B[k], c1, col[1]);
      col[2] = fmaf(B[k], c2, col[2]);
    }
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

int launch_preprocess(gs_ctx* ctx, cudaStream_t s) {
  const int64_t N = ctx->N;
  if (N == 0) return GS_OK;
  const int threads = 128;  // 64 registers, 8 CTAs / SM: the kernel is latency-bound (measured 256x3: 34.0, 256x4: 31.6, 128x8: 30.9, 128x10: 34.5 us)
  const unsigned blocks = (unsigned)div_up(N, threads);
#define GS_PRE(D)                                                                                                    \
  GS_LAUNCH_PDL(preprocess_kernel<D>, blocks, threads, 0, s, N, ctx->means, ctx->scales, ctx->quats, ctx->opacities, \
                ctx->sh, ctx->cam, ctx->feat, ctx->tiles_touched, ctx->tile_count, ctx->vis_ids, ctx->vis_rec,        \
                ctx->vis_par, ctx->slot_of, ctx->counts, ctx->pose_acc)
  switch (ctx->sh_degree) {
    case 0: GS_PRE(0); break;
    case 1: GS_PRE(1); break;
    case 2: GS_PRE(2); break;
    default: GS_PRE(3); break;
  }
#undef GS_PRE
  GS_LAUNCH_CHECK("preprocess_kernel");
  return GS_OK;
}

}  // namespace gs

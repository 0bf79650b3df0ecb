// gs_gauss_bwd.cu -- step a9 (per-Gaussian chain rule: 2-D gradients -> mu, s, q, opacity, SH) and step a10 (6-DoF
// pose gradient: block-reduced partial sums, then a one-thread final kernel).  One thread per visible Gaussian for the
// arithmetic; every row-shaped transfer (the SH row in, the gradient rows out) is done by the whole CTA through shared
// memory so that consecutive lanes touch consecutive 16 bytes (one thread per row meant 32 different 128-byte lines per
// load / store instruction: the kernel sat on the L1 tag stage and on its 128 registers, profiles/r2_stages.md).
// HBM-bound (gradient rows of (11 + 3K) floats per Gaussian).
#include "gs_internal.cuh"
#include "gs_project.cuh"
#include "gs_raster.cuh"
#include "gs_sh.cuh"

namespace gs {

// scalar type of the per-Gaussian chain: fp32 (the gradient tolerance is 1e-3 relative L2; the forward projection in
// gs_preprocess stays fp64).  The pose partial sums are reduced in fp32 inside a warp and in fp64 beyond.
using R = float;
__device__ __forceinline__ float gs_rsqrt(float x) { return rsqrtf(x); }
__device__ __forceinline__ double gs_rsqrt(double x) { return rsqrt(x); }

// GS_ACCUMULATE adds into the caller's arrays with fire-and-forget reductions at L2 (RED.ADD.F32, 16 bytes at a time for
// the SH rows): a load + add + store chained a DRAM round trip into every step of the store loops (config 5: 206 us per
// view).  A row belongs to one Gaussian and is touched once per launch, so the result is the same single fp32 addition.
__device__ __forceinline__ void store_or_add(float* p, float v, bool accumulate) {
  if (accumulate) atomicAdd(p, v); else *p = v;
}

// DEG: SH degree.  WRITE: parameter gradients are produced (false = GS_POSE_ONLY).
#ifndef GS_GB_MIN_CTAS
#define GS_GB_MIN_CTAS 5
#endif
template <int DEG, bool WRITE>
__global__ void __launch_bounds__(128, GS_GB_MIN_CTAS)
gauss_bwd_kernel(int64_t N, const float* __restrict__ means, const float* __restrict__ scales,
                 const float* __restrict__ quats, const float* __restrict__ opacities, const float* __restrict__ sh,
                 DevCam cam, const uint32_t* __restrict__ vis_ids, const float4* __restrict__ vis_par,
                 const float4* __restrict__ feat, const Counts* __restrict__ counts,
                 const uint32_t* __restrict__ tiles_touched, float* __restrict__ g2d, bool accumulate, bool sparse, bool fill,
                 float* __restrict__ g_means, float* __restrict__ g_scales, float* __restrict__ g_quats,
                 float* __restrict__ g_opac, float* __restrict__ g_sh, double* __restrict__ pose_acc) {
  constexpr int K = (DEG + 1) * (DEG + 1);
  // one thread per VISIBLE Gaussian (compacted list of gs_preprocess)
  const int64_t kk = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  pdl_enter();
  const uint32_t V = counts->n_visible;
  if (WRITE && fill) {
    // Dense outputs: exact zeros for the culled Gaussians.  Block b clears the culled rows among the Gaussians
    // [128 b, 128 b + 128) -- N - V rows in total instead of a memset of all N (the five cudaMemsetAsync on a side stream
    // cost raster_bwd 23 us of the SMs they ran on, profiles/r2_stages.md); the rows of the visible Gaussians are written
    // below by the blocks that own their visible slots.  Rows are cleared by consecutive threads in 16-byte pieces.
    __shared__ uint32_t s_rows[128];
    __shared__ uint32_t s_wcnt[4];
    const bool culled = kk < N && tiles_touched[kk] == 0u;
    const unsigned bal = __ballot_sync(0xffffffffu, culled);
    const int wl = threadIdx.x >> 5, ln = threadIdx.x & 31;
    if (ln == 0) s_wcnt[wl] = __popc(bal);
    __syncthreads();
    uint32_t before = 0, cnt = 0;
#pragma unroll
    for (int w = 0; w < 4; ++w) { before += w < wl ? s_wcnt[w] : 0u; cnt += s_wcnt[w]; }
    if (culled) s_rows[before + __popc(bal & ((1u << ln) - 1u))] = (uint32_t)kk;
    __syncthreads();
    const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
    if constexpr ((3 * K) % 4 == 0) {
      constexpr int Q = 3 * K / 4;  // float4 per SH row
      for (uint32_t t = threadIdx.x; t < cnt * Q; t += blockDim.x) {
        const uint32_t r = t / Q, c = t - r * Q;
        reinterpret_cast<float4*>(g_sh + (int64_t)3 * K * s_rows[r])[c] = z4;
      }
    } else {
      for (uint32_t t = threadIdx.x; t < cnt * (3 * K); t += blockDim.x) {
        const uint32_t r = t / (3 * K), c = t - r * (3 * K);
        g_sh[(int64_t)3 * K * s_rows[r] + c] = 0.f;
      }
    }
    for (uint32_t t = threadIdx.x; t < cnt * 3; t += blockDim.x) {
      const uint32_t r = t / 3, c = t - r * 3;
      g_means[(int64_t)3 * s_rows[r] + c] = 0.f;
      g_scales[(int64_t)3 * s_rows[r] + c] = 0.f;
    }
    for (uint32_t t = threadIdx.x; t < cnt; t += blockDim.x) {
      reinterpret_cast<float4*>(g_quats)[s_rows[t]] = z4;
      g_opac[s_rows[t]] = 0.f;
    }
  }
  const int64_t blk0 = (int64_t)blockIdx.x * blockDim.x;
  if (blk0 >= (int64_t)V) return;
  // ---- rows of this block: SH rows in (cp.async, whole CTA), gradient rows out (whole CTA) -------------------------
  // Row layout in shared memory: 3K floats at a stride of RS floats chosen so that one thread per row reads its row
  // without bank conflicts (float4 accesses when 3K % 4 == 0: 12 -> stride 12, 48 -> stride 52; scalar otherwise: odd 3K).
  constexpr int K3 = 3 * K;
  constexpr bool V4 = (K3 % 4) == 0;
  constexpr int RS = V4 ? ((K3 / 4) % 2 ? K3 : K3 + 4) : K3;
  constexpr int EW = V4 ? 4 : 1, EPR = K3 / EW;  // floats per element, elements per row
  __shared__ __align__(16) float s_sh[128 * RS];
  __shared__ __align__(16) float s_small[128 * 11];  // g_mean (3), g_scale (3), g_quat (4), g_opacity (1) per row
  __shared__ uint32_t s_ids[128];
  const int tid = threadIdx.x;
  const int nrow = (int)min((int64_t)128, (int64_t)V - blk0);
  const bool vis = tid < nrow;
  const int64_t i = vis ? (int64_t)vis_ids[kk] : 0;
  s_ids[tid] = (uint32_t)i;
  __syncthreads();
  for (int f = tid; f < nrow * EPR; f += 128) {
    const int r = f / EPR, c = f - r * EPR;
    const float* src = sh + (int64_t)K3 * s_ids[r] + c * EW;
    if constexpr (V4) cp_async16(s_sh + r * RS + c * EW, src); else cp_async4(s_sh + r * RS + c * EW, src);
  }
  float T[12];
  load_pose(cam, T);
  R acc[15];
#pragma unroll
  for (int k = 0; k < 15; ++k) acc[k] = (R)0;
  R gpc[3] = {0, 0, 0};
  R Wm[9];
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) Wm[3 * r + c] = T[4 * r + c];
  float gcol[3] = {0.f, 0.f, 0.f};
  float mu0 = 0.f, mu1 = 0.f, mu2 = 0.f;
  float* sm = s_small + tid * 11;
  if (vis) {
    // g2d and the parameter copies are stored by visible slot (= this thread's index): sequential streams
    float4* gp4 = reinterpret_cast<float4*>(g2d + (size_t)kk * kG2D);
    const float4 ga = gp4[0], gb = gp4[1], gc = gp4[2];
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    gp4[0] = zero; gp4[1] = zero; gp4[2] = zero;  // keep the accumulator all-zero for the next iteration
    const float4 pa = __ldg(vis_par + 3 * (size_t)kk), pb = __ldg(vis_par + 3 * (size_t)kk + 1), q = __ldg(vis_par + 3 * (size_t)kk + 2);
    mu0 = pa.x; mu1 = pa.y; mu2 = pa.z;
    const float o = pa.w;
    const float s0 = pb.x, s1 = pb.y, s2 = pb.z;
    Proj<R> P;
    project_gaussian<R, false>(cam, T, mu0, mu1, mu2, s0, s1, s2, q.x, q.y, q.z, q.w, o, P);
    // 2-D gradients from the whitened moments (gs_internal.cuh): with k Q = L L^T and w = L^T d,
    //   dL/dmean = sum gp Q d = L M1 / k,      dL/dSigma' = sum gp (Q d)(Q d)^T / 2 = L M2 L^T / (2 k^2);
    // L comes from the forward's feature record (fp64 Cholesky in gs_preprocess), so neither the fp32 determinant of
    // Sigma' nor the product -Q gQ Q (which cancels for long thin footprints) is ever formed here.
    const R* W = Wm;
    const float4 f1 = __ldg(feat + 3 * (size_t)kk + 1);
    const R l11 = f1.x, l21 = f1.y, l22 = f1.z;
    const R ik = (R)(2.0 * 0.69314718055994531);  // 1 / k, k = 0.5 log2(e)
    const R g_mx = ik * l11 * (R)ga.x, g_my = ik * (l21 * (R)ga.x + l22 * (R)ga.y);
    const R g_o = (R)gb.y / (R)o;
    gcol[0] = gb.z; gcol[1] = gb.w; gcol[2] = gc.x;
    const R g_z = gc.y;
    const R hk = (R)0.5 * ik * ik;
    const R n00 = l11 * (R)ga.z, n01 = l11 * (R)ga.w;
    const R n10 = l21 * (R)ga.z + l22 * (R)ga.w, n11 = l21 * (R)ga.w + l22 * (R)gb.x;
    const R gS00 = hk * n00 * l11, gS01 = hk * (n00 * l21 + n01 * l22), gS10 = gS01, gS11 = hk * (n10 * l21 + n11 * l22);
    // gM = 2 gS M
    R gM[6];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      gM[c] = (R)2.0 * (gS00 * P.M[c] + gS01 * P.M[3 + c]);
      gM[3 + c] = (R)2.0 * (gS10 * P.M[c] + gS11 * P.M[3 + c]);
    }
    // gT = gM M3^T ; gM3 = Tm^T gM
    R gT[6], gM3[9];
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
      for (int c = 0; c < 3; ++c)
        gT[3 * r + c] = gM[3 * r] * P.M3[3 * c] + gM[3 * r + 1] * P.M3[3 * c + 1] + gM[3 * r + 2] * P.M3[3 * c + 2];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
      for (int c = 0; c < 3; ++c) gM3[3 * r + c] = P.Tm[r] * gM[c] + P.Tm[3 + r] * gM[3 + c];
    // M3 = R diag(s)
    const R sd[3] = {s0, s1, s2};
    R gR[9];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      sm[3 + c] = (float)(P.Rm[c] * gM3[c] + P.Rm[3 + c] * gM3[3 + c] + P.Rm[6 + c] * gM3[6 + c]);  // g_scale
#pragma unroll
      for (int r = 0; r < 3; ++r) gR[3 * r + c] = gM3[3 * r + c] * sd[c];
    }
    // quaternion (w,x,y,z): gr_k = <gR, dR/dr_k>, then through the normalisation
    const R w = P.r[0], x = P.r[1], y = P.r[2], z = P.r[3];
    R gr[4];
    gr[0] = (R)2.0 * (-z * gR[1] + y * gR[2] + z * gR[3] - x * gR[5] - y * gR[6] + x * gR[7]);
    gr[1] = (R)2.0 * (y * gR[1] + z * gR[2] + y * gR[3] - (R)2.0 * x * gR[4] - w * gR[5] + z * gR[6] + w * gR[7] - (R)2.0 * x * gR[8]);
    gr[2] = (R)2.0 * (-(R)2.0 * y * gR[0] + x * gR[1] + w * gR[2] + x * gR[3] + z * gR[5] - w * gR[6] + z * gR[7] - (R)2.0 * y * gR[8]);
    gr[3] = (R)2.0 * (-(R)2.0 * z * gR[0] - w * gR[1] + x * gR[2] + w * gR[3] - (R)2.0 * z * gR[4] + y * gR[5] + x * gR[6] + y * gR[7]);
    const R rd = w * gr[0] + x * gr[1] + y * gr[2] + z * gr[3];
    const R iqn = (R)1.0 / P.qn;
#pragma unroll
    for (int k = 0; k < 4; ++k) sm[6 + k] = (float)((gr[k] - P.r[k] * rd) * iqn);  // g_quat
    sm[10] = (float)g_o;
    // T = J W: gJ = gT W^T (only the four non-zero entries of J), gW += J^T gT
    const R gJ00 = gT[0] * W[0] + gT[1] * W[1] + gT[2] * W[2];
    const R gJ02 = gT[0] * W[6] + gT[1] * W[7] + gT[2] * W[8];
    const R gJ11 = gT[3] * W[3] + gT[4] * W[4] + gT[5] * W[5];
    const R gJ12 = gT[3] * W[6] + gT[4] * W[7] + gT[5] * W[8];
    const R iz = (R)1.0 / P.z, iz2 = iz * iz, fx = cam.fx, fy = cam.fy;
    gpc[0] = g_mx * fx * iz - gJ02 * fx * iz2;
    gpc[1] = g_my * fy * iz - gJ12 * fy * iz2;
    gpc[2] = -g_mx * fx * P.x * iz2 - g_my * fy * P.y * iz2 + g_z - gJ00 * fx * iz2 - gJ11 * fy * iz2 +
             (R)2.0 * gJ02 * fx * P.x * iz2 * iz + (R)2.0 * gJ12 * fy * P.y * iz2 * iz;
    // pose partial sums: sum g_pc, sum g_v (below), g_W = J^T gT + g_pc mu^T
    acc[0] = gpc[0]; acc[1] = gpc[1]; acc[2] = gpc[2];
    const R mud[3] = {mu0, mu1, mu2};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      acc[6 + c] = P.J00 * gT[c] + gpc[0] * mud[c];
      acc[9 + c] = P.J11 * gT[3 + c] + gpc[1] * mud[c];
      acc[12 + c] = P.J02 * gT[c] + P.J12 * gT[3 + c] + gpc[2] * mud[c];
    }
  }
  cp_async_wait_all();
  __syncthreads();  // the SH rows of the block have landed
  if (vis) {
    const R* W = Wm;
    // colour: same fp32 sequence as the forward, so the clamp decision is identical
    const R ccx = -((R)T[0] * T[3] + (R)T[4] * T[7] + (R)T[8] * T[11]);
    const R ccy = -((R)T[1] * T[3] + (R)T[5] * T[7] + (R)T[9] * T[11]);
    const R ccz = -((R)T[2] * T[3] + (R)T[6] * T[7] + (R)T[10] * T[11]);
    const R vx = (R)mu0 - ccx, vy = (R)mu1 - ccy, vz = (R)mu2 - ccz;
    const R ivn = gs_rsqrt(vx * vx + vy * vy + vz * vz);
    const float nx = (float)(vx * ivn), ny = (float)(vy * ivn), nz = (float)(vz * ivn);
    float B[K];
    sh_basis<DEG>(nx, ny, nz, B);
    float* row = s_sh + tid * RS;
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
    float gcr[3];
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) gcr[ch] = (col[ch] + 0.5f > 0.f) ? gcol[ch] : 0.f;
    // second pass over the row: w_k = <sh_k, g_craw> for the view-direction gradient; the row is overwritten in place by
    // the SH gradient B_k g_craw
    float wk[K];
#pragma unroll
    for (int k = 0; k < K; ++k) wk[k] = 0.f;
    if constexpr (V4) {
#pragma unroll
      for (int v = 0; v < K3 / 4; ++v) {
        float4* p4 = reinterpret_cast<float4*>(row + 4 * v);
        const float4 t = *p4;
        const float e[4] = {t.x, t.y, t.z, t.w};
        float g[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          wk[(4 * v + u) / 3] = fmaf(e[u], gcr[(4 * v + u) % 3], wk[(4 * v + u) / 3]);
          g[u] = B[(4 * v + u) / 3] * gcr[(4 * v + u) % 3];
        }
        if (WRITE) *p4 = make_float4(g[0], g[1], g[2], g[3]);
      }
    } else {
#pragma unroll
      for (int k = 0; k < K3; ++k) {
        wk[k / 3] = fmaf(row[k], gcr[k % 3], wk[k / 3]);
        if (WRITE) row[k] = B[k / 3] * gcr[k % 3];
      }
    }
    float gnx = 0.f, gny = 0.f, gnz = 0.f;
    if (DEG > 0) sh_basis_grad<DEG>(nx, ny, nz, wk, gnx, gny, gnz);
    const R nd = (R)nx * gnx + (R)ny * gny + (R)nz * gnz;
    const R gv[3] = {((R)gnx - nx * nd) * ivn, ((R)gny - ny * nd) * ivn, ((R)gnz - nz * nd) * ivn};
    acc[3] = gv[0]; acc[4] = gv[1]; acc[5] = gv[2];
#pragma unroll
    for (int c = 0; c < 3; ++c) sm[c] = (float)(W[c] * gpc[0] + W[3 + c] * gpc[1] + W[6 + c] * gpc[2] + gv[c]);  // g_mean
  }
  if (WRITE) {
    __syncthreads();
    // gradient rows leave by the whole CTA: consecutive threads write consecutive elements of a row.  Output row of
    // block-row r: GS_SPARSE_GRADS writes one row per VISIBLE Gaussian in slot order, else the row of Gaussian s_ids[r].
    for (int f = tid; f < nrow * EPR; f += 128) {
      const int r = f / EPR, c = f - r * EPR;
      const int64_t orow = sparse ? blk0 + r : (int64_t)s_ids[r];
      float* dst = g_sh + (int64_t)K3 * orow + c * EW;
      if constexpr (V4) {
        float4 val = *reinterpret_cast<const float4*>(s_sh + r * RS + c * EW);
        if (accumulate) atomicAdd(reinterpret_cast<float4*>(dst), val); else *reinterpret_cast<float4*>(dst) = val;
      } else {
        store_or_add(dst, s_sh[r * RS + c], accumulate);
      }
    }
    for (int f = tid; f < nrow * 3; f += 128) {
      const int r = f / 3, c = f - r * 3;
      const int64_t orow = sparse ? blk0 + r : (int64_t)s_ids[r];
      store_or_add(g_means + 3 * orow + c, s_small[r * 11 + c], accumulate);
      store_or_add(g_scales + 3 * orow + c, s_small[r * 11 + 3 + c], accumulate);
    }
    for (int f = tid; f < nrow * 4; f += 128) {
      const int r = f >> 2, c = f & 3;
      const int64_t orow = sparse ? blk0 + r : (int64_t)s_ids[r];
      store_or_add(g_quats + 4 * orow + c, s_small[r * 11 + 6 + c], accumulate);
    }
    if (vis) store_or_add(g_opac + (sparse ? kk : i), s_small[tid * 11 + 10], accumulate);
  }
  // block reduction of the 15 pose partials: fp32 inside the warp, fp64 across warps and blocks, one atomic set per block
  __shared__ double s_acc[4][15];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool any = __any_sync(0xffffffffu, vis);
  if (any) {
#pragma unroll
    for (int k = 0; k < 15; ++k) {
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) acc[k] += __shfl_xor_sync(0xffffffffu, acc[k], d);
    }
  }
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < 15; ++k) s_acc[warp][k] = any ? (double)acc[k] : 0.0;
  }
  __syncthreads();
  if (threadIdx.x < 15) {
    const double v = s_acc[0][threadIdx.x] + s_acc[1][threadIdx.x] + s_acc[2][threadIdx.x] + s_acc[3][threadIdx.x];
    if (v != 0.0) atomicAdd(pose_acc + threadIdx.x, v);
  }
}

// g_rho = sum g_pc + W sum g_v ; g_phi_k = <g_W, [e_k]x W> + (sum g_pc) . (e_k x t)      (C4)
__global__ void pose_final_kernel(DevCam cam, const double* __restrict__ pose_acc, bool accumulate,
                                  float* __restrict__ g_twist) {
  pdl_enter();
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  float T[12];
  load_pose(cam, T);
  const double W[9] = {T[0], T[1], T[2], T[4], T[5], T[6], T[8], T[9], T[10]};
  const double t[3] = {T[3], T[7], T[11]};
  const double* gpc = pose_acc;
  const double* gv = pose_acc + 3;
  const double* gW = pose_acc + 6;
  double out[6];
  for (int r = 0; r < 3; ++r) out[r] = gpc[r] + W[3 * r] * gv[0] + W[3 * r + 1] * gv[1] + W[3 * r + 2] * gv[2];
  for (int k = 0; k < 3; ++k) {
    const int k1 = (k + 1) % 3, k2 = (k + 2) % 3;
    // ([e_k]x W) has row k1 = -W row k2 ... written out: (e_k x v)_k1 = -v_k2, (e_k x v)_k2 = v_k1
    double a = 0.0;
    for (int c = 0; c < 3; ++c) a += gW[3 * k2 + c] * W[3 * k1 + c] - gW[3 * k1 + c] * W[3 * k2 + c];
    a += gpc[k2] * t[k1] - gpc[k1] * t[k2];
    out[3 + k] = a;
  }
  for (int k = 0; k < 6; ++k) g_twist[k] = accumulate ? g_twist[k] + (float)out[k] : (float)out[k];
}

int launch_gauss_bwd(gs_ctx* ctx, cudaStream_t s, uint32_t flags, float* g_means, float* g_scales, float* g_quats,
                     float* g_opac, float* g_sh) {
  if (!ctx->pose_acc_clean) GS_CUDA(cudaMemsetAsync(ctx->pose_acc, 0, 15 * sizeof(double), s));
  ctx->pose_acc_clean = false;
  ctx->pose_acc_valid = true;
  ctx->g2d_dirty = false;
  if (ctx->N == 0) return GS_OK;
  const bool write = !(flags & GS_POSE_ONLY);
  const bool accum = (flags & GS_ACCUMULATE) != 0;
  const bool sparse = (flags & GS_SPARSE_GRADS) != 0;
  const bool fill = write && !accum && !sparse;  // dense outputs: the kernel clears the rows of the culled Gaussians itself
  const int threads = 128;
  const unsigned blocks = (unsigned)div_up(ctx->N, threads);
#define GS_GB(D, Wr)                                                                                                 \
  GS_LAUNCH_PDL((gauss_bwd_kernel<D, Wr>), blocks, threads, 0, s, ctx->N, ctx->means, ctx->scales, ctx->quats,      \
                ctx->opacities, ctx->sh, ctx->cam, (const uint32_t*)ctx->vis_ids, (const float4*)ctx->vis_par,        \
                (const float4*)ctx->feat, (const Counts*)ctx->counts, (const uint32_t*)ctx->tiles_touched, ctx->g2d,  \
                accum, sparse, fill, g_means, g_scales, g_quats, g_opac, g_sh, ctx->pose_acc)
  if (write) {
    switch (ctx->sh_degree) {
      case 0: GS_GB(0, true); break;
      case 1: GS_GB(1, true); break;
      case 2: GS_GB(2, true); break;
      default: GS_GB(3, true); break;
    }
  } else {
    switch (ctx->sh_degree) {
      case 0: GS_GB(0, false); break;
      case 1: GS_GB(1, false); break;
      case 2: GS_GB(2, false); break;
      default: GS_GB(3, false); break;
    }
  }
#undef GS_GB
  GS_LAUNCH_CHECK("gauss_bwd_kernel");
  return GS_OK;
}

int launch_pose_final(gs_ctx* ctx, cudaStream_t s, uint32_t flags, float* g_twist) {
  GS_LAUNCH_PDL(pose_final_kernel, 1, 32, 0, s, ctx->cam, (const double*)ctx->pose_acc, (flags & GS_ACCUMULATE) != 0, g_twist);
  GS_LAUNCH_CHECK("pose_final_kernel");
  return GS_OK;
}

}  // namespace gs

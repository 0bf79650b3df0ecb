// gs_sh.cuh -- real spherical harmonics (degree 0..3) for the CUDA path: basis values and their gradient w.r.t. the
// unit direction.  Ordering l = 0..3, m = -l..l; real form with the (-1)^m sign convention (Q10).
#pragma once

namespace gs {

// 1/(2 sqrt(pi)); sqrt(3/(4 pi)); {1/2 sqrt(15/pi), 1/4 sqrt(5/pi), 1/4 sqrt(15/pi)};
// {1/4 sqrt(35/(2 pi)), 1/2 sqrt(105/pi), 1/4 sqrt(21/(2 pi)), 1/4 sqrt(7/pi), 1/4 sqrt(105/pi)}
#define GS_SH0 0.28209479177387814f
#define GS_SH1 0.4886025119029199f
#define GS_SH2A 1.0925484305920792f
#define GS_SH2B 0.31539156525252005f
#define GS_SH2C 0.5462742152960396f
#define GS_SH3A 0.5900435899266435f
#define GS_SH3B 2.890611442640554f
#define GS_SH3C 0.4570457994644658f
#define GS_SH3D 0.3731763325901154f
#define GS_SH3E 1.445305721320277f

template <int DEG>
__device__ __forceinline__ void sh_basis(float x, float y, float z, float* B) {
  B[0] = GS_SH0;
  if (DEG >= 1) {
    B[1] = -GS_SH1 * y;
    B[2] = GS_SH1 * z;
    B[3] = -GS_SH1 * x;
  }
  if (DEG >= 2) {
    const float xx = x * x, yy = y * y, zz = z * z;
    B[4] = GS_SH2A * x * y;
    B[5] = -GS_SH2A * y * z;
    B[6] = GS_SH2B * (2.f * zz - xx - yy);
    B[7] = -GS_SH2A * x * z;
    B[8] = GS_SH2C * (xx - yy);
    if (DEG >= 3) {
      B[9] = -GS_SH3A * y * (3.f * xx - yy);
      B[10] = GS_SH3B * x * y * z;
      B[11] = -GS_SH3C * y * (4.f * zz - xx - yy);
      B[12] = GS_SH3D * z * (2.f * zz - 3.f * xx - 3.f * yy);
      B[13] = -GS_SH3C * x * (4.f * zz - xx - yy);
      B[14] = GS_SH3E * z * (xx - yy);
      B[15] = -GS_SH3A * x * (xx - 3.f * yy);
    }
  }
}

// Accumulates g_n += sum_k (dB_k/dn) * w_k, w_k = <sh_k, g_craw>.
template <int DEG>
__device__ __forceinline__ void sh_basis_grad(float x, float y, float z, const float* w, float& gx, float& gy,
                                              float& gz) {
  gx = gy = gz = 0.f;
  if (DEG >= 1) {
    gy += -GS_SH1 * w[1];
    gz += GS_SH1 * w[2];
    gx += -GS_SH1 * w[3];
  }
  if (DEG >= 2) {
    gx += GS_SH2A * y * w[4];
    gy += GS_SH2A * x * w[4];
    gy += -GS_SH2A * z * w[5];
    gz += -GS_SH2A * y * w[5];
    gx += -2.f * GS_SH2B * x * w[6];
    gy += -2.f * GS_SH2B * y * w[6];
    gz += 4.f * GS_SH2B * z * w[6];
    gx += -GS_SH2A * z * w[7];
    gz += -GS_SH2A * x * w[7];
    gx += 2.f * GS_SH2C * x * w[8];
    gy += -2.f * GS_SH2C * y * w[8];
  }
  if (DEG >= 3) {
    const float xx = x * x, yy = y * y, zz = z * z;
    gx += -GS_SH3A * 6.f * x * y * w[9];
    gy += -GS_SH3A * (3.f * xx - 3.f * yy) * w[9];
    gx += GS_SH3B * y * z * w[10];
    gy += GS_SH3B * x * z * w[10];
    gz += GS_SH3B * x * y * w[10];
    gx += GS_SH3C * 2.f * x * y * w[11];
    gy += -GS_SH3C * (4.f * zz - xx - 3.f * yy) * w[11];
    gz += -GS_SH3C * 8.f * y * z * w[11];
    gx += -GS_SH3D * 6.f * x * z * w[12];
    gy += -GS_SH3D * 6.f * y * z * w[12];
    gz += GS_SH3D * (6.f * zz - 3.f * xx - 3.f * yy) * w[12];
    gx += -GS_SH3C * (4.f * zz - 3.f * xx - yy) * w[13];
    gy += GS_SH3C * 2.f * x * y * w[13];
    gz += -GS_SH3C * 8.f * x * z * w[13];
    gx += GS_SH3E * 2.f * x * z * w[14];
    gy += -GS_SH3E * 2.f * y * z * w[14];
    gz += GS_SH3E * (xx - yy) * w[14];
    gx += -GS_SH3A * (3.f * xx - 3.f * yy) * w[15];
    gy += GS_SH3A * 6.f * x * y * w[15];
  }
}

}  // namespace gs

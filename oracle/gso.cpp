// gso.cpp -- ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).
//
// A plain, slow, fp64 CPU statement of what the hot path computes: differentiable 3D Gaussian Splatting rendering of
// RGB, depth and alpha (Eq. 4 "I^, D^"; "the differentiably rendered RGB and depth") and its
// analytic gradients w.r.t. every Gaussian parameter (mu, s, q, opacity, colour; Eq. 19)
// and the world-to-camera keyframe pose ("per-keyframe pose deltas").
//
// The paper is silent on the rasteriser's internals; the constants and conventions are the readings C1-C5 / Q1-Q17
// listed in DESIGN.md ("Readings of the paper").  The forward is the plain per-pixel ordered sum (no tiles, no
// blocking); the backward is the plain chain rule, written in the order of DESIGN.md's formulas.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call this library.  It
// shares no code, header, table or constant with paper_2605_10760_b200/csrc (the CUDA path) and never includes it.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): quaternion vs Rodrigues/scipy; SH orthonormality by quadrature and
// scipy.special; EWA closed form + Monte-Carlo; single-Gaussian closed-form image; occlusion; monotone transmittance;
// central finite differences of every gradient incl. pose; rigid/scale covariance (Eq. 19 + Eq. 15); brute-force
// rendering without boxes; brute-force binning.  Parity unpinned: none of the functions; the *choice* among readings
// Q3, Q5, Q6, Q8 is a convention.
//
// Build: g++ -O2 -fopenmp -shared -fPIC (oracle/build.py).  -ffast-math is NOT used.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

struct gso_camera {
  int32_t width, height;
  double fx, fy, cx, cy, near_z;
  double T_cw[12];  // row-major [R|t], p_c = R p_w + t
};

struct gso_options {
  double dilation;    // 0.3   (Q4)
  double alpha_min;   // 1/255 (Q1)   0 disables the test
  double alpha_max;   // 0.99  (Q2)   +inf disables the clamp
  double T_min;       // 1e-4  (Q3)   0 disables the early exit
  int32_t tile;       // 16
  int32_t brute_force;  // 1: every pixel visits every visible Gaussian (no bounding boxes)
  int32_t max_threads;  // 0 = all
  int32_t reserved;
};

}  // extern "C"

namespace {

const double kPi = 3.14159265358979323846;

// ---------------------------------------------------------------------------------------------------------------
// Real spherical harmonics, degree 0..3, on the unit vector n = (x,y,z); order l = 0..3, m = -l..l (reading C1.5).
// Constants are computed from their closed forms.  dB[k*3+j] = d B_k / d n_j of the polynomial written here.
// ---------------------------------------------------------------------------------------------------------------
void sh_basis(int deg, const double n[3], double B[16], double dB[48]) {
  const double x = n[0], y = n[1], z = n[2];
  for (int k = 0; k < 16; ++k) { B[k] = 0; dB[3 * k] = dB[3 * k + 1] = dB[3 * k + 2] = 0; }
  auto set = [&](int k, double v, double dx, double dy, double dz) {
    B[k] = v; dB[3 * k] = dx; dB[3 * k + 1] = dy; dB[3 * k + 2] = dz;
  };
  set(0, 1.0 / (2.0 * std::sqrt(kPi)), 0, 0, 0);
  if (deg < 1) return;
  const double c1 = std::sqrt(3.0 / (4.0 * kPi));
  set(1, -c1 * y, 0, -c1, 0);
  set(2, c1 * z, 0, 0, c1);
  set(3, -c1 * x, -c1, 0, 0);
  if (deg < 2) return;
  const double c2a = 0.5 * std::sqrt(15.0 / kPi), c2b = 0.25 * std::sqrt(5.0 / kPi), c2c = 0.25 * std::sqrt(15.0 / kPi);
  set(4, c2a * x * y, c2a * y, c2a * x, 0);
  set(5, -c2a * y * z, 0, -c2a * z, -c2a * y);
  set(6, c2b * (2 * z * z - x * x - y * y), -2 * c2b * x, -2 * c2b * y, 4 * c2b * z);
  set(7, -c2a * x * z, -c2a * z, 0, -c2a * x);
  set(8, c2c * (x * x - y * y), 2 * c2c * x, -2 * c2c * y, 0);
  if (deg < 3) return;
  const double c3a = 0.25 * std::sqrt(35.0 / (2.0 * kPi)), c3b = 0.5 * std::sqrt(105.0 / kPi),
               c3c = 0.25 * std::sqrt(21.0 / (2.0 * kPi)), c3d = 0.25 * std::sqrt(7.0 / kPi),
               c3e = 0.25 * std::sqrt(105.0 / kPi);
  set(9, -c3a * y * (3 * x * x - y * y), -c3a * 6 * x * y, -c3a * (3 * x * x - 3 * y * y), 0);
  set(10, c3b * x * y * z, c3b * y * z, c3b * x * z, c3b * x * y);
  set(11, -c3c * y * (4 * z * z - x * x - y * y), c3c * 2 * x * y, -c3c * (4 * z * z - x * x - 3 * y * y),
      -c3c * 8 * y * z);
  set(12, c3d * z * (2 * z * z - 3 * x * x - 3 * y * y), -c3d * 6 * x * z, -c3d * 6 * y * z,
      c3d * (6 * z * z - 3 * x * x - 3 * y * y));
  set(13, -c3c * x * (4 * z * z - x * x - y * y), -c3c * (4 * z * z - 3 * x * x - y * y), c3c * 2 * x * y,
      -c3c * 8 * x * z);
  set(14, c3e * z * (x * x - y * y), c3e * 2 * x * z, -c3e * 2 * y * z, c3e * (x * x - y * y));
  set(15, -c3a * x * (x * x - 3 * y * y), -c3a * (3 * x * x - 3 * y * y), c3a * 6 * x * y, 0);
}

// Unit quaternion r = (w,x,y,z) -> rotation matrix (row-major), reading Q11.
void quat_to_R(const double r[4], double R[9]) {
  const double w = r[0], x = r[1], y = r[2], z = r[3];
  R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - w * z);     R[2] = 2 * (x * z + w * y);
  R[3] = 2 * (x * y + w * z);     R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - w * x);
  R[6] = 2 * (x * z - w * y);     R[7] = 2 * (y * z + w * x);     R[8] = 1 - 2 * (x * x + y * y);
}

// <gR, dR/dr_k>, k = w,x,y,z, for the polynomial above.
void quat_R_backward(const double r[4], const double gR[9], double gr[4]) {
  const double w = r[0], x = r[1], y = r[2], z = r[3];
  const double dW[9] = {0, -z, y, z, 0, -x, -y, x, 0};
  const double dX[9] = {0, y, z, y, -2 * x, -w, z, w, -2 * x};
  const double dY[9] = {-2 * y, x, w, x, 0, z, -w, z, -2 * y};
  const double dZ[9] = {-2 * z, -w, x, w, -2 * z, y, x, y, 0};
  gr[0] = gr[1] = gr[2] = gr[3] = 0;
  for (int k = 0; k < 9; ++k) {
    gr[0] += 2 * gR[k] * dW[k]; gr[1] += 2 * gR[k] * dX[k]; gr[2] += 2 * gR[k] * dY[k]; gr[3] += 2 * gR[k] * dZ[k];
  }
}

// Everything the forward computes for one Gaussian (reading C1, steps 1-6 and 8).
struct Proj {
  bool visible;
  double pc[3];          // camera-space centre (x,y,z)
  double rq[4], qnorm;   // unit quaternion and |q|
  double R[9], M3[9];    // R(r), M3 = R diag(s)
  double J[6], Tm[6], M[6];  // J (2x3), T = J W (2x3), M = T M3 (2x3)
  double cov[3];         // Sigma' = M M^T + dilation I : xx, xy, yy
  double con[3];         // Q = Sigma'^-1 : a, b, c
  double m[2];           // pixel-space centre (integer-centred pixels, Q7)
  double v[3], vnorm, n[3];  // view vector mu - c_cam, its norm, unit direction
  double B[16], dB[48];
  double craw[3], col[3];  // SH sum + 0.5 ; max(0, .)
  float z32;             // canonical fp32 depth key (C1.6)
  double hx, hy;         // exact half extents of {alpha >= alpha_min} (Q5 (ii)); inf if alpha_min == 0
  int32_t px[4];         // pixel span [x0,x1) x [y0,y1)  -> order x0,y0,x1,y1
  int32_t tl[4];         // tile span  [tx0,tx1) x [ty0,ty1)
};

inline int32_t clamp_to_int(double v, int32_t lo, int32_t hi) {
  if (!(v > (double)lo)) return lo;
  if (!(v < (double)hi)) return hi;
  return (int32_t)v;
}

// Parameters arrive as doubles: the float32 arrays the GPU path receives, promoted exactly by the caller (or genuinely
// fp64 values in the finite-difference tests).
void project(int deg, const double* mu, const double* s, const double* q32, double o, const double* sh32,
             const gso_camera& cam, const gso_options& opt, Proj& P) {
  const double* Tcw = cam.T_cw;
  const double W[9] = {Tcw[0], Tcw[1], Tcw[2], Tcw[4], Tcw[5], Tcw[6], Tcw[8], Tcw[9], Tcw[10]};
  const double t[3] = {Tcw[3], Tcw[7], Tcw[11]};
  P.visible = false;
  for (int k = 0; k < 4; ++k) P.px[k] = P.tl[k] = 0;
  // 1. camera space + near cull + opacity cull
  for (int r = 0; r < 3; ++r) P.pc[r] = W[3 * r] * mu[0] + W[3 * r + 1] * mu[1] + W[3 * r + 2] * mu[2] + t[r];
  const double x = P.pc[0], y = P.pc[1], z = P.pc[2];
  // 6. canonical fp32 depth key
  {
    const float W20 = (float)Tcw[8], W21 = (float)Tcw[9], W22 = (float)Tcw[10], tz = (float)Tcw[11];
    P.z32 = std::fmaf(W20, (float)mu[0], std::fmaf(W21, (float)mu[1], std::fmaf(W22, (float)mu[2], tz)));
  }
  if (!(z > cam.near_z)) return;
  if (o < opt.alpha_min) return;
  // 2. covariance factor
  double qn = std::sqrt(q32[0] * q32[0] + q32[1] * q32[1] + q32[2] * q32[2] + q32[3] * q32[3]);
  P.qnorm = qn;
  for (int k = 0; k < 4; ++k) P.rq[k] = q32[k] / qn;
  quat_to_R(P.rq, P.R);
  for (int r = 0; r < 3; ++r)
    for (int c = 0; c < 3; ++c) P.M3[3 * r + c] = P.R[3 * r + c] * s[c];
  // 3. EWA projection
  P.J[0] = cam.fx / z; P.J[1] = 0;          P.J[2] = -cam.fx * x / (z * z);
  P.J[3] = 0;          P.J[4] = cam.fy / z; P.J[5] = -cam.fy * y / (z * z);
  for (int r = 0; r < 2; ++r)
    for (int c = 0; c < 3; ++c)
      P.Tm[3 * r + c] = P.J[3 * r] * W[c] + P.J[3 * r + 1] * W[3 + c] + P.J[3 * r + 2] * W[6 + c];
  for (int r = 0; r < 2; ++r)
    for (int c = 0; c < 3; ++c)
      P.M[3 * r + c] = P.Tm[3 * r] * P.M3[c] + P.Tm[3 * r + 1] * P.M3[3 + c] + P.Tm[3 * r + 2] * P.M3[6 + c];
  P.cov[0] = P.M[0] * P.M[0] + P.M[1] * P.M[1] + P.M[2] * P.M[2] + opt.dilation;
  P.cov[1] = P.M[0] * P.M[3] + P.M[1] * P.M[4] + P.M[2] * P.M[5];
  P.cov[2] = P.M[3] * P.M[3] + P.M[4] * P.M[4] + P.M[5] * P.M[5] + opt.dilation;
  const double det = P.cov[0] * P.cov[2] - P.cov[1] * P.cov[1];
  if (!(det > 0) || !std::isfinite(det)) return;
  P.con[0] = P.cov[2] / det; P.con[1] = -P.cov[1] / det; P.con[2] = P.cov[0] / det;
  // 4. pixel-space centre
  P.m[0] = cam.fx * x / z + cam.cx;
  P.m[1] = cam.fy * y / z + cam.cy;
  if (!std::isfinite(P.m[0]) || !std::isfinite(P.m[1])) return;
  // 5. colour
  const double ccam[3] = {-(W[0] * t[0] + W[3] * t[1] + W[6] * t[2]), -(W[1] * t[0] + W[4] * t[1] + W[7] * t[2]),
                          -(W[2] * t[0] + W[5] * t[1] + W[8] * t[2])};
  for (int k = 0; k < 3; ++k) P.v[k] = mu[k] - ccam[k];
  P.vnorm = std::sqrt(P.v[0] * P.v[0] + P.v[1] * P.v[1] + P.v[2] * P.v[2]);
  for (int k = 0; k < 3; ++k) P.n[k] = P.v[k] / P.vnorm;
  sh_basis(deg, P.n, P.B, P.dB);
  const int K = (deg + 1) * (deg + 1);
  for (int ch = 0; ch < 3; ++ch) {
    double acc = 0;
    for (int k = 0; k < K; ++k) acc += P.B[k] * sh32[3 * k + ch];
    P.craw[ch] = acc + 0.5;
    P.col[ch] = acc + 0.5 > 0 ? acc + 0.5 : 0.0;
  }
  // 8. exact extent of {alpha >= alpha_min}: d^T Q d <= rho^2 = 2 ln(o / alpha_min); bbox half widths rho sqrt(cov)
  const int32_t Wd = cam.width, Ht = cam.height, ts = opt.tile;
  if (opt.alpha_min > 0) {
    const double rho = std::sqrt(2.0 * std::log(o / opt.alpha_min));
    P.hx = rho * std::sqrt(P.cov[0]);
    P.hy = rho * std::sqrt(P.cov[2]);
    P.px[0] = clamp_to_int(std::ceil(P.m[0] - P.hx), 0, Wd);
    P.px[1] = clamp_to_int(std::ceil(P.m[1] - P.hy), 0, Ht);
    P.px[2] = clamp_to_int(std::floor(P.m[0] + P.hx) + 1.0, 0, Wd);
    P.px[3] = clamp_to_int(std::floor(P.m[1] + P.hy) + 1.0, 0, Ht);
  } else {
    P.hx = P.hy = std::numeric_limits<double>::infinity();
    P.px[0] = 0; P.px[1] = 0; P.px[2] = Wd; P.px[3] = Ht;
  }
  if (P.px[2] <= P.px[0] || P.px[3] <= P.px[1]) return;
  P.tl[0] = P.px[0] / ts; P.tl[1] = P.px[1] / ts;
  P.tl[2] = (P.px[2] - 1) / ts + 1; P.tl[3] = (P.px[3] - 1) / ts + 1;
  P.visible = true;
}

inline uint32_t float_bits(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }

int num_threads(const gso_options& opt) {
#ifdef _OPENMP
  int n = omp_get_max_threads();
  if (n > 64) n = 64;
  if (opt.max_threads > 0 && opt.max_threads < n) n = opt.max_threads;
  return n < 1 ? 1 : n;
#else
  (void)opt; return 1;
#endif
}

}  // namespace

extern "C" {

int gso_num_threads(const gso_options* opt) { return num_threads(*opt); }

void gso_default_options(gso_options* o) {
  o->dilation = 0.3; o->alpha_min = 1.0 / 255.0; o->alpha_max = 0.99; o->T_min = 1e-4; o->tile = 16;
  o->brute_force = 0; o->max_threads = 0; o->reserved = 0;
}

// --- small exported pieces, so the tests can pin them one by one -------------------------------------------------
void gso_sh_basis(int deg, const double* n, double* B, double* dB) { sh_basis(deg, n, B, dB); }
void gso_quat_to_R(const double* q, double* R) {
  double qn = std::sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
  double r[4] = {q[0] / qn, q[1] / qn, q[2] / qn, q[3] / qn};
  quat_to_R(r, R);
}

// Exp(xi^) for xi = (rho, phi): R = I + A K + B K^2, t = V rho, V = I + B K + C K^2 (reading C4).
void gso_se3_exp(const double* xi, double* R, double* t) {
  const double* rho = xi; const double* phi = xi + 3;
  const double th2 = phi[0] * phi[0] + phi[1] * phi[1] + phi[2] * phi[2], th = std::sqrt(th2);
  double A, Bc, C;
  if (th < 1e-6) { A = 1 - th2 / 6; Bc = 0.5 - th2 / 24; C = 1.0 / 6 - th2 / 120; }
  else { A = std::sin(th) / th; Bc = (1 - std::cos(th)) / th2; C = (th - std::sin(th)) / (th2 * th); }
  const double K[9] = {0, -phi[2], phi[1], phi[2], 0, -phi[0], -phi[1], phi[0], 0};
  double K2[9];
  for (int r = 0; r < 3; ++r)
    for (int c = 0; c < 3; ++c) K2[3 * r + c] = K[3 * r] * K[c] + K[3 * r + 1] * K[3 + c] + K[3 * r + 2] * K[6 + c];
  for (int k = 0; k < 9; ++k) R[k] = (k % 4 == 0 ? 1.0 : 0.0) + A * K[k] + Bc * K2[k];
  for (int r = 0; r < 3; ++r) {
    t[r] = 0;
    for (int c = 0; c < 3; ++c) t[r] += ((r == c ? 1.0 : 0.0) + Bc * K[3 * r + c] + C * K2[3 * r + c]) * rho[c];
  }
}

// T_out = Exp(xi^) T_in  (left-multiplicative twist on the world-to-camera pose, reading Q14).
void gso_pose_apply(const double* xi, const double* T_in, double* T_out) {
  double R[9], tv[3];
  gso_se3_exp(xi, R, tv);
  for (int r = 0; r < 3; ++r) {
    for (int c = 0; c < 3; ++c)
      T_out[4 * r + c] = R[3 * r] * T_in[c] + R[3 * r + 1] * T_in[4 + c] + R[3 * r + 2] * T_in[8 + c];
    T_out[4 * r + 3] = R[3 * r] * T_in[3] + R[3 * r + 1] * T_in[7] + R[3 * r + 2] * T_in[11] + tv[r];
  }
}

// ---------------------------------------------------------------------------------------------------------------
// gso_preprocess: reading C1 steps 1-6, 8.  All outputs are caller-owned host arrays; any may be null.
//   visible u8[N]; pc f64[N,3]; mean2d f64[N,2]; cov2d f64[N,3]; conic f64[N,3]; rgb f64[N,3] (after clamp);
//   z f64[N] (= pc.z); z32 f32[N]; rect_px i32[N,4] (x0,y0,x1,y1 half-open); rect_tile i32[N,4].
// ---------------------------------------------------------------------------------------------------------------
int gso_preprocess(int64_t N, int sh_degree, const double* means, const double* scales, const double* quats,
                   const double* opacities, const double* sh, const gso_camera* cam, const gso_options* opt,
                   uint8_t* visible, double* pc, double* mean2d, double* cov2d, double* conic, double* rgb,
                   double* z, float* z32, int32_t* rect_px, int32_t* rect_tile) {
  if (sh_degree < 0 || sh_degree > 3 || N < 0) return -1;
  const int K = (sh_degree + 1) * (sh_degree + 1);
#pragma omp parallel for schedule(static) num_threads(num_threads(*opt))
  for (int64_t i = 0; i < N; ++i) {
    Proj P;
    std::memset(&P, 0, sizeof(P));
    project(sh_degree, means + 3 * i, scales + 3 * i, quats + 4 * i, opacities[i], sh + 3 * (int64_t)K * i, *cam,
            *opt, P);
    if (visible) visible[i] = P.visible ? 1 : 0;
    if (z32) z32[i] = P.z32;
    if (z) z[i] = P.pc[2];
    if (pc) for (int k = 0; k < 3; ++k) pc[3 * i + k] = P.pc[k];
    for (int k = 0; k < 4; ++k) {
      if (rect_px) rect_px[4 * i + k] = P.visible ? P.px[k] : 0;
      if (rect_tile) rect_tile[4 * i + k] = P.visible ? P.tl[k] : 0;
    }
    for (int k = 0; k < 3; ++k) {
      if (cov2d) cov2d[3 * i + k] = P.visible ? P.cov[k] : 0;
      if (conic) conic[3 * i + k] = P.visible ? P.con[k] : 0;
      if (rgb) rgb[3 * i + k] = P.visible ? P.col[k] : 0;
    }
    if (mean2d) { mean2d[2 * i] = P.visible ? P.m[0] : 0; mean2d[2 * i + 1] = P.visible ? P.m[1] : 0; }
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------------------------
// gso_bin: reading C1 step 8 / Q13.  Integer only.  Given per-Gaussian tile rects [tx0,tx1) x [ty0,ty1) (an empty rect
// emits nothing) and depth keys z32: instances (tile = ty*tiles_x + tx, bits(z32), i), ordered by (tile, bits, i);
// ranges[t] = [first, last+1).  Returns the instance count; fills keys/ids only if capacity suffices (null = count).
// ---------------------------------------------------------------------------------------------------------------
int64_t gso_bin(int64_t N, const int32_t* rect_tile, const float* z32, int32_t tiles_x, int32_t tiles_y,
                int64_t capacity, uint64_t* keys, uint32_t* ids, uint32_t* ranges) {
  struct Inst { uint64_t key; uint32_t id; };
  std::vector<Inst> v;
  for (int64_t i = 0; i < N; ++i) {
    const int32_t* r = rect_tile + 4 * i;
    for (int32_t ty = r[1]; ty < r[3]; ++ty)
      for (int32_t tx = r[0]; tx < r[2]; ++tx) {
        if (tx < 0 || ty < 0 || tx >= tiles_x || ty >= tiles_y) return -1;
        uint64_t tile = (uint64_t)ty * (uint64_t)tiles_x + (uint64_t)tx;
        v.push_back({(tile << 32) | (uint64_t)float_bits(z32[i]), (uint32_t)i});
      }
  }
  std::stable_sort(v.begin(), v.end(), [](const Inst& a, const Inst& b) {
    if (a.key != b.key) return a.key < b.key;
    return a.id < b.id;
  });
  const int64_t I = (int64_t)v.size();
  if (keys && ids && capacity >= I)
    for (int64_t k = 0; k < I; ++k) { keys[k] = v[k].key; ids[k] = v[k].id; }
  if (ranges) {
    const int64_t T = (int64_t)tiles_x * tiles_y;
    for (int64_t t = 0; t < 2 * T; ++t) ranges[t] = 0;
    for (int64_t k = 0; k < I; ++k) {
      const uint64_t tile = v[k].key >> 32;
      if (k == 0 || (v[k - 1].key >> 32) != tile) ranges[2 * tile] = (uint32_t)k;
      if (k == I - 1 || (v[k + 1].key >> 32) != tile) ranges[2 * tile + 1] = (uint32_t)(k + 1);
    }
  }
  return I;
}

// ---------------------------------------------------------------------------------------------------------------
// gso_render: reading C1 step 7 (forward) and C2 (per-pixel backward, if d_rgb != null).
// Inputs are the per-Gaussian features in fp64 (from gso_preprocess, or hand-built by a test) + z32 for the order.
// Forward outputs: rgb f64[3,H,W], depth f64[H,W], alpha f64[H,W], n_blended i32[H,W], margin f64[H,W] (C6).
// Backward outputs (accumulated from zero): g_mean2d[N,2], g_conic[N,3] (a,b,c), g_opac[N], g_rgb[N,3], g_z[N].
// The box used to skip Gaussians is the exact extent (hx,hy recomputed here from cov2d and opacity) padded by
// 0.1 % + 1e-3 px; outside it alpha < alpha_min, so the result is the definition's; brute_force=1 drops the boxes.
// ---------------------------------------------------------------------------------------------------------------
int gso_render(int64_t N, const uint8_t* visible, const double* mean2d, const double* cov2d, const double* conic,
               const double* opacities, const double* rgb_g, const double* z, const float* z32,
               const gso_camera* cam, const gso_options* opt, const double* bg,
               double* out_rgb, double* out_depth, double* out_alpha, int32_t* out_nblend, double* out_margin,
               const double* d_rgb, const double* d_depth, const double* d_alpha,
               double* g_mean2d, double* g_conic, double* g_opac, double* g_rgb, double* g_z) {
  const int32_t Wd = cam->width, Ht = cam->height;
  const int64_t HW = (int64_t)Wd * Ht;
  // global order pi: visible Gaussians by (bits(z32), index)
  std::vector<int64_t> order;
  for (int64_t i = 0; i < N; ++i) if (visible[i]) order.push_back(i);
  std::stable_sort(order.begin(), order.end(), [&](int64_t a, int64_t b) {
    const uint32_t ka = float_bits(z32[a]), kb = float_bits(z32[b]);
    if (ka != kb) return ka < kb;
    return a < b;
  });
  const int64_t V = (int64_t)order.size();
  // padded pixel boxes [bx0,bx1) x [by0,by1)
  std::vector<int32_t> bx0(V), bx1(V), by0(V), by1(V);
  for (int64_t k = 0; k < V; ++k) {
    const int64_t i = order[k];
    if (opt->brute_force || !(opt->alpha_min > 0)) { bx0[k] = 0; by0[k] = 0; bx1[k] = Wd; by1[k] = Ht; continue; }
    const double rho = std::sqrt(2.0 * std::log(opacities[i] / opt->alpha_min));
    const double hx = rho * std::sqrt(cov2d[3 * i]) * 1.001 + 1e-3, hy = rho * std::sqrt(cov2d[3 * i + 2]) * 1.001 + 1e-3;
    bx0[k] = clamp_to_int(std::ceil(mean2d[2 * i] - hx), 0, Wd);
    by0[k] = clamp_to_int(std::ceil(mean2d[2 * i + 1] - hy), 0, Ht);
    bx1[k] = clamp_to_int(std::floor(mean2d[2 * i] + hx) + 1.0, 0, Wd);
    by1[k] = clamp_to_int(std::floor(mean2d[2 * i + 1] + hy) + 1.0, 0, Ht);
  }
  // per-row candidate lists, in order pi
  std::vector<std::vector<int32_t>> rows(Ht);
  for (int64_t k = 0; k < V; ++k)
    for (int32_t y = by0[k]; y < by1[k]; ++y) rows[y].push_back((int32_t)k);

  const bool bwd = d_rgb != nullptr;
  const int nt = num_threads(*opt);
  std::vector<std::vector<double>> acc;  // per-thread [V,10]: gm(2) gcon(3) go(1) grgb(3) gz(1)
  if (bwd) acc.assign(nt, std::vector<double>());

#pragma omp parallel num_threads(nt)
  {
#ifdef _OPENMP
    const int tid = omp_get_thread_num();
#else
    const int tid = 0;
#endif
    double* A = nullptr;
    if (bwd) { acc[tid].assign((size_t)V * 10, 0.0); A = acc[tid].data(); }
    struct Rec { int32_t k; double alpha, T, dx, dy, G; bool clamped; };
    std::vector<Rec> recs;
#pragma omp for schedule(static, 1)  // interleaved rows: balanced, and the summation order is reproducible
    for (int32_t py = 0; py < Ht; ++py) {
      const std::vector<int32_t>& cand = rows[py];
      for (int32_t px = 0; px < Wd; ++px) {
        recs.clear();
        double T = 1.0, C[3] = {0, 0, 0}, D = 0, margin = std::numeric_limits<double>::infinity();
        for (int32_t k : cand) {
          if (px < bx0[k] || px >= bx1[k]) continue;
          const int64_t i = order[k];
          const double dx = (double)px - mean2d[2 * i], dy = (double)py - mean2d[2 * i + 1];
          const double a = conic[3 * i], b = conic[3 * i + 1], c = conic[3 * i + 2];
          const double power = -0.5 * (a * dx * dx + c * dy * dy) - b * dx * dy;
          if (power > 0) continue;
          const double G = std::exp(power);
          const double oG = opacities[i] * G;
          const double alpha = oG < opt->alpha_max ? oG : opt->alpha_max;
          if (opt->alpha_min > 0) margin = std::min(margin, std::fabs(alpha / opt->alpha_min - 1.0));
          if (alpha < opt->alpha_min) continue;
          if (opt->T_min > 0) margin = std::min(margin, std::fabs(T / opt->T_min - 1.0));
          if (T < opt->T_min) break;  // Q3 (b): i is blended iff the transmittance in front of it is >= T_min
          recs.push_back({k, alpha, T, dx, dy, G, oG > opt->alpha_max});
          const double w = alpha * T;
          for (int ch = 0; ch < 3; ++ch) C[ch] += rgb_g[3 * i + ch] * w;
          D += z[i] * w;
          T *= (1.0 - alpha);
        }
        const int64_t p = (int64_t)py * Wd + px;
        if (out_rgb) for (int ch = 0; ch < 3; ++ch) out_rgb[ch * HW + p] = C[ch] + T * bg[ch];
        if (out_depth) out_depth[p] = D;
        if (out_alpha) out_alpha[p] = 1.0 - T;
        if (out_nblend) out_nblend[p] = (int32_t)recs.size();
        if (out_margin) out_margin[p] = margin;
        if (!bwd) continue;
        // C2: back-to-front
        const double gC[3] = {d_rgb[p], d_rgb[HW + p], d_rgb[2 * HW + p]};
        const double gD = d_depth ? d_depth[p] : 0.0, gA = d_alpha ? d_alpha[p] : 0.0;
        double S = T * (gC[0] * bg[0] + gC[1] * bg[1] + gC[2] * bg[2]);
        for (int64_t r = (int64_t)recs.size() - 1; r >= 0; --r) {
          const Rec& e = recs[r];
          const int64_t i = order[e.k];
          double* g = A + (size_t)e.k * 10;
          const double wgt = e.alpha * e.T;
          const double w_i = gC[0] * rgb_g[3 * i] + gC[1] * rgb_g[3 * i + 1] + gC[2] * rgb_g[3 * i + 2] + gD * z[i] + gA;
          for (int ch = 0; ch < 3; ++ch) g[6 + ch] += wgt * gC[ch];
          g[9] += wgt * gD;
          const double dalpha = e.T * w_i - S / (1.0 - e.alpha);
          S += w_i * wgt;
          if (e.clamped) continue;  // Q2: no flow to opacity / G through the clamp
          g[5] += e.G * dalpha;
          const double gG = opacities[i] * dalpha * e.G;  // dL/dpower
          const double a = conic[3 * i], b = conic[3 * i + 1], c = conic[3 * i + 2];
          g[0] += gG * (a * e.dx + b * e.dy);
          g[1] += gG * (b * e.dx + c * e.dy);
          g[2] += gG * (-0.5 * e.dx * e.dx);
          g[3] += gG * (-e.dx * e.dy);
          g[4] += gG * (-0.5 * e.dy * e.dy);
        }
      }
    }
  }
  if (bwd) {
    for (int64_t i = 0; i < N; ++i) {
      if (g_mean2d) g_mean2d[2 * i] = g_mean2d[2 * i + 1] = 0;
      if (g_conic) g_conic[3 * i] = g_conic[3 * i + 1] = g_conic[3 * i + 2] = 0;
      if (g_opac) g_opac[i] = 0;
      if (g_rgb) g_rgb[3 * i] = g_rgb[3 * i + 1] = g_rgb[3 * i + 2] = 0;
      if (g_z) g_z[i] = 0;
    }
    for (int64_t k = 0; k < V; ++k) {
      const int64_t i = order[k];
      double s[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
      for (int t = 0; t < nt; ++t) {
        if (acc[t].empty()) continue;
        for (int j = 0; j < 10; ++j) s[j] += acc[t][(size_t)k * 10 + j];
      }
      if (g_mean2d) { g_mean2d[2 * i] = s[0]; g_mean2d[2 * i + 1] = s[1]; }
      if (g_conic) { g_conic[3 * i] = s[2]; g_conic[3 * i + 1] = s[3]; g_conic[3 * i + 2] = s[4]; }
      if (g_opac) g_opac[i] = s[5];
      if (g_rgb) { g_rgb[3 * i] = s[6]; g_rgb[3 * i + 1] = s[7]; g_rgb[3 * i + 2] = s[8]; }
      if (g_z) g_z[i] = s[9];
    }
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------------------------
// gso_preprocess_bwd: reading C3 (per-Gaussian chain rule) and C4 (pose gradient).
// Inputs: the parameters, the camera, and the 2D gradients from gso_render.  Outputs (dense, zeros for culled):
// g_means[N,3], g_scales[N,3], g_quats[N,4], g_opacities[N], g_sh[N,K,3], g_twist[6] = (rho, phi), and optionally the
// raw sums g_W[9], g_pc_sum[3], g_v_sum[3] (for the tests of C4).
// ---------------------------------------------------------------------------------------------------------------
int gso_preprocess_bwd(int64_t N, int sh_degree, const double* means, const double* scales, const double* quats,
                       const double* opacities, const double* sh, const gso_camera* cam, const gso_options* opt,
                       const double* g_mean2d, const double* g_conic, const double* g_opac_in, const double* g_rgb,
                       const double* g_z, double* g_means, double* g_scales, double* g_quats, double* g_opacities,
                       double* g_sh, double* g_twist, double* out_gW, double* out_gpc_sum, double* out_gv_sum) {
  if (sh_degree < 0 || sh_degree > 3) return -1;
  const int K = (sh_degree + 1) * (sh_degree + 1);
  const double* Tcw = cam->T_cw;
  const double W[9] = {Tcw[0], Tcw[1], Tcw[2], Tcw[4], Tcw[5], Tcw[6], Tcw[8], Tcw[9], Tcw[10]};
  const double t[3] = {Tcw[3], Tcw[7], Tcw[11]};
  double gW[9] = {0}, gpc_sum[3] = {0}, gv_sum[3] = {0};
  for (int64_t i = 0; i < N; ++i) {
    Proj P;
    std::memset(&P, 0, sizeof(P));
    project(sh_degree, means + 3 * i, scales + 3 * i, quats + 4 * i, opacities[i], sh + 3 * (int64_t)K * i, *cam,
            *opt, P);
    double gmu[3] = {0, 0, 0}, gs[3] = {0, 0, 0}, gq[4] = {0, 0, 0, 0}, go = 0;
    if (g_sh) for (int k = 0; k < 3 * K; ++k) g_sh[3 * (int64_t)K * i + k] = 0;
    if (P.visible) {
      const double x = P.pc[0], y = P.pc[1], z = P.pc[2], fx = cam->fx, fy = cam->fy;
      const double mu[3] = {means[3 * i], means[3 * i + 1], means[3 * i + 2]};
      const double s[3] = {scales[3 * i], scales[3 * i + 1], scales[3 * i + 2]};
      go = g_opac_in[i];
      // conic -> Sigma'
      const double ga = g_conic[3 * i], gb = g_conic[3 * i + 1], gc = g_conic[3 * i + 2];
      const double Q[4] = {P.con[0], P.con[1], P.con[1], P.con[2]};
      const double gQ[4] = {ga, 0.5 * gb, 0.5 * gb, gc};
      double QgQ[4], gS[4];
      for (int r = 0; r < 2; ++r)
        for (int c = 0; c < 2; ++c) QgQ[2 * r + c] = Q[2 * r] * gQ[c] + Q[2 * r + 1] * gQ[2 + c];
      for (int r = 0; r < 2; ++r)
        for (int c = 0; c < 2; ++c) gS[2 * r + c] = -(QgQ[2 * r] * Q[c] + QgQ[2 * r + 1] * Q[2 + c]);
      // Sigma' = M M^T + dil I  ->  g_M = 2 g_Sigma' M
      double gM[6];
      for (int r = 0; r < 2; ++r)
        for (int c = 0; c < 3; ++c) gM[3 * r + c] = 2.0 * (gS[2 * r] * P.M[c] + gS[2 * r + 1] * P.M[3 + c]);
      // M = T M3 -> g_T = g_M M3^T (2x3), g_M3 = T^T g_M (3x3)
      double gT[6], gM3[9];
      for (int r = 0; r < 2; ++r)
        for (int c = 0; c < 3; ++c)
          gT[3 * r + c] = gM[3 * r] * P.M3[3 * c] + gM[3 * r + 1] * P.M3[3 * c + 1] + gM[3 * r + 2] * P.M3[3 * c + 2];
      for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) gM3[3 * r + c] = P.Tm[r] * gM[c] + P.Tm[3 + r] * gM[3 + c];
      // M3 = R diag(s)
      double gR[9];
      for (int c = 0; c < 3; ++c) {
        gs[c] = P.R[c] * gM3[c] + P.R[3 + c] * gM3[3 + c] + P.R[6 + c] * gM3[6 + c];
        for (int r = 0; r < 3; ++r) gR[3 * r + c] = gM3[3 * r + c] * s[c];
      }
      double gr[4];
      quat_R_backward(P.rq, gR, gr);
      const double rdot = P.rq[0] * gr[0] + P.rq[1] * gr[1] + P.rq[2] * gr[2] + P.rq[3] * gr[3];
      for (int k = 0; k < 4; ++k) gq[k] = (gr[k] - P.rq[k] * rdot) / P.qnorm;
      // T = J W -> g_J = g_T W^T (2x3), g_W += J^T g_T
      double gJ[6];
      for (int r = 0; r < 2; ++r)
        for (int c = 0; c < 3; ++c) gJ[3 * r + c] = gT[3 * r] * W[3 * c] + gT[3 * r + 1] * W[3 * c + 1] + gT[3 * r + 2] * W[3 * c + 2];
      for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) gW[3 * r + c] += P.J[r] * gT[c] + P.J[3 + r] * gT[3 + c];
      // camera-space centre
      const double gmx = g_mean2d[2 * i], gmy = g_mean2d[2 * i + 1];
      double gpc[3];
      gpc[0] = gmx * fx / z + gJ[2] * (-fx / (z * z));
      gpc[1] = gmy * fy / z + gJ[5] * (-fy / (z * z));
      gpc[2] = -gmx * fx * x / (z * z) - gmy * fy * y / (z * z) + g_z[i] + gJ[0] * (-fx / (z * z)) +
               gJ[4] * (-fy / (z * z)) + gJ[2] * (2 * fx * x / (z * z * z)) + gJ[5] * (2 * fy * y / (z * z * z));
      // colour
      double gcraw[3];
      for (int ch = 0; ch < 3; ++ch) gcraw[ch] = P.craw[ch] > 0 ? g_rgb[3 * i + ch] : 0.0;
      double gn[3] = {0, 0, 0};
      for (int k = 0; k < K; ++k) {
        double shg = 0;
        for (int ch = 0; ch < 3; ++ch) {
          if (g_sh) g_sh[3 * ((int64_t)K * i + k) + ch] = P.B[k] * gcraw[ch];
          shg += sh[3 * ((int64_t)K * i + k) + ch] * gcraw[ch];
        }
        for (int j = 0; j < 3; ++j) gn[j] += P.dB[3 * k + j] * shg;
      }
      const double ndot = P.n[0] * gn[0] + P.n[1] * gn[1] + P.n[2] * gn[2];
      double gv[3];
      for (int j = 0; j < 3; ++j) gv[j] = (gn[j] - P.n[j] * ndot) / P.vnorm;
      // p_c = W mu + t
      for (int j = 0; j < 3; ++j) gmu[j] = W[j] * gpc[0] + W[3 + j] * gpc[1] + W[6 + j] * gpc[2] + gv[j];
      for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) gW[3 * r + c] += gpc[r] * mu[c];
      for (int j = 0; j < 3; ++j) { gpc_sum[j] += gpc[j]; gv_sum[j] += gv[j]; }
    }
    if (g_means) for (int j = 0; j < 3; ++j) g_means[3 * i + j] = gmu[j];
    if (g_scales) for (int j = 0; j < 3; ++j) g_scales[3 * i + j] = gs[j];
    if (g_quats) for (int j = 0; j < 4; ++j) g_quats[4 * i + j] = gq[j];
    if (g_opacities) g_opacities[i] = go;
  }
  // C4: g_rho = sum g_pc + W sum g_v ; g_phi_k = <g_W, [e_k]x W> + (sum g_pc) . (e_k x t)
  if (g_twist) {
    for (int r = 0; r < 3; ++r) g_twist[r] = gpc_sum[r] + W[3 * r] * gv_sum[0] + W[3 * r + 1] * gv_sum[1] + W[3 * r + 2] * gv_sum[2];
    for (int k = 0; k < 3; ++k) {
      double e[3] = {0, 0, 0}; e[k] = 1;
      const double Kx[9] = {0, -e[2], e[1], e[2], 0, -e[0], -e[1], e[0], 0};
      double acc2 = 0;
      for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) {
          const double KW = Kx[3 * r] * W[c] + Kx[3 * r + 1] * W[3 + c] + Kx[3 * r + 2] * W[6 + c];
          acc2 += gW[3 * r + c] * KW;
        }
      const double ext[3] = {e[1] * t[2] - e[2] * t[1], e[2] * t[0] - e[0] * t[2], e[0] * t[1] - e[1] * t[0]};
      acc2 += gpc_sum[0] * ext[0] + gpc_sum[1] * ext[1] + gpc_sum[2] * ext[2];
      g_twist[3 + k] = acc2;
    }
  }
  if (out_gW) for (int k = 0; k < 9; ++k) out_gW[k] = gW[k];
  if (out_gpc_sum) for (int k = 0; k < 3; ++k) out_gpc_sum[k] = gpc_sum[k];
  if (out_gv_sum) for (int k = 0; k < 3; ++k) out_gv_sum[k] = gv_sum[k];
  return 0;
}

}  // extern "C"

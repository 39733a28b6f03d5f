// =====================================================================================
//  SSS-GS forward relighting render path -- CPU ORACLE (test infrastructure only).
//
//  This file is TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and the
//  `cpu_baseline` / `--impl reference` legs of bench.py may load it.  The product
//  (libsssgs.so, paper_2408_12282_b200/csrc) shares no code with it and never calls it.
//
//  It is a plain, slow, step-by-step restatement of what the path computes, written
//  from /root/reference/PAPER.md ("L<n>" = line n of that file) with the readings
//  S1..S19 of SURVEY.md 8(c) where the paper is silent (each listed in DESIGN.md).
//  Arithmetic is double precision, except the projection (step 3) which is the
//  "canonical fp32 sequence" P1..P10: sort keys and tile rectangles depend on it and
//  must be bit-exact on both sides, so it is defined operation by operation in IEEE
//  binary32 (compile with -ffp-contract=off; fmaf() is a single rounding).
//
//  Parity status of the readings that cannot be pinned from the paper
//  ("parity unpinned"): S1 (which 2 rotation components feed the MLP),
//  S8 (choice of D/F/G lobes and the factor 4 in Eq. 4), S10 (coverage normalisation
//  before shading), and the ray rule of orc_bake_visibility (the paper only says rays are
//  traced "similar to [10]": where along the ray a Gaussian acts, the opacity rule and the
//  ray offset t_min are this build's reading; its arithmetic IS pinned).
//  Every function below is otherwise pinned by tests/test_oracle_*.py
//  against closed forms, invariants, library special cases or brute force.
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---- constants (the paper inherits them from the kernels of [18], L138) ----
constexpr double kAlphaMin = 1.0 / 255.0;  // skip a Gaussian at a pixel if alpha < 1/255
constexpr double kAlphaMax = 0.99;         // alpha clamp
constexpr double kTMin = 1e-4;             // stop when transmittance would drop below this
constexpr float kLowPass = 0.3f;           // screen-space low-pass added to Sigma' diagonal
constexpr float kFrustumClamp = 1.3f;      // clamp of x/z, y/z used in the Jacobian only
constexpr float kDiscFloor = 0.1f;         // floor of the eigenvalue discriminant
constexpr float kRadiusSigma = 3.33f;      // K_R >= sqrt(2 ln 255) (S3: image is tile independent)
constexpr double kPi = 3.14159265358979323846;
constexpr double kY00 = 0.2820948;         // real SH basis constants (S14)
constexpr double kY1 = 0.4886025;
constexpr int kGbufChannels = 16;

enum { ACT_RELU = 0, ACT_LEAKY_RELU = 1 };

inline double round_bf16(double v) {
  // value -> float32 -> bf16 (round to nearest even) -> double
  float f = (float)v;
  uint32_t u;
  std::memcpy(&u, &f, 4);
  if ((u & 0x7F800000u) == 0x7F800000u) return (double)f;  // inf / nan unchanged
  uint32_t lsb = (u >> 16) & 1u;
  u = (u + 0x7FFFu + lsb) & 0xFFFF0000u;
  std::memcpy(&f, &u, 4);
  return (double)f;
}

// value -> float32 -> IEEE binary16 (round to nearest even, subnormals kept, finite overflow
// saturates to +-65504 as the kernel's cvt.rn.satfinite does) -> double.  Written from the format's
// definition: the binary16 numbers of a binade [2^(e-1), 2^e) are spaced q = 2^(e-1-10) apart, q is
// 2^-24 below the smallest normal 2^-14; x / q is exact (a power-of-two scaling) and nearbyint rounds
// it to the nearest integer, ties to even (default rounding mode).
inline double round_fp16(double v) {
  const float f = (float)v;
  if (std::isnan(f)) return (double)f;
  const double a = std::fabs((double)f);
  if (a > 65504.0) return std::copysign(65504.0, (double)f);  // includes +-inf (satfinite)
  if (a == 0.0) return (double)f;
  int e;
  std::frexp(a, &e);  // a = m 2^e, m in [0.5, 1)
  const int eq = (e - 1 < -14 ? -14 : e - 1) - 10;
  const double q = std::ldexp(1.0, eq);
  const double r = std::nearbyint(a / q) * q;
  return std::copysign(r > 65504.0 ? 65504.0 : r, (double)f);
}

}  // namespace

extern "C" {

// The two rounding helpers, exposed so that tests can pin them against independent library
// conversions (torch bfloat16, numpy float16).
void orc_round_bf16(int64_t n, const double* in, double* out) {
  for (int64_t i = 0; i < n; ++i) out[i] = round_bf16(in[i]);
}
void orc_round_fp16(int64_t n, const double* in, double* out) {
  for (int64_t i = 0; i < n; ++i) out[i] = round_fp16(in[i]);
}

// Camera as passed by the tests (mirrors the fields of sssgs_camera, include/sssgs.h).
struct OrcCamera {
  float R[9];
  float t[3];
  float fx, fy, cx, cy, tan_half_fovx, tan_half_fovy;
  int width, height;
  float znear;
  float bg[3];
};

int orc_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// -------------------------------------------------------------------------------------
// Step 1 -- MLP input assembly.  PAPER.md L98 Eq. 6: f(mu, Sigma, n, w_in, w_out, v);
// L347: "(16+24) feature dimensions, with normals (3), rotation (2), scale (3), light
// direction (3), view direction (3), light distance (1) and visibility (1).  The position
// (3) is encoded using a positional Fourier encoding [27] resulting in 24 features."
// Row layout (in L347's order of enumeration):
//   x = [ n(3) | rot(2) | scale(3) | w_in(3) | w_out(3) | d(1) | v(1) | gamma(mu)(24) | feat(F) ]
//   rot   = (q_w, q_x) of the sign-canonicalised (q_w >= 0) unit quaternion          (S1)
//   w_in  = (p_L - mu)/|.|, w_out = (p_cam - mu)/|.|, d = |p_L - mu|                  (S15)
//   v     = clamp(sum_lm c_lm Y_lm(w_in), 0, 1), Y_00 = .2820948, Y_1{-1,0,1} = .4886025{y,z,x} (S14)
//   gamma = for k = 0..3: [sin(2^k pi mu_xyz), cos(2^k pi mu_xyz)]                     (S13)
// p_cam = -R^T t.
// -------------------------------------------------------------------------------------
void orc_mlp_inputs(int64_t n, const float* means, const float* normals, const float* rotations,
                    const float* scales, const float* vis_sh, int sh_degree, const float* feat,
                    int F, const OrcCamera* cam, const float* light_pos, double* x_out) {
  const int D = 40 + F;
  double pc[3];
  for (int k = 0; k < 3; ++k)
    pc[k] = -((double)cam->R[0 + k] * cam->t[0] + (double)cam->R[3 + k] * cam->t[1] +
              (double)cam->R[6 + k] * cam->t[2]);
  const int ncoef = (sh_degree + 1) * (sh_degree + 1);
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double* x = x_out + i * D;
    const double mu[3] = {means[3 * i], means[3 * i + 1], means[3 * i + 2]};
    for (int k = 0; k < 3; ++k) x[k] = normals[3 * i + k];
    double sgn = rotations[4 * i] < 0.f ? -1.0 : 1.0;
    x[3] = sgn * rotations[4 * i];
    x[4] = sgn * rotations[4 * i + 1];
    for (int k = 0; k < 3; ++k) x[5 + k] = scales[3 * i + k];
    double wi[3], wo[3], di = 0, dn = 0;
    for (int k = 0; k < 3; ++k) {
      wi[k] = (double)light_pos[k] - mu[k];
      wo[k] = pc[k] - mu[k];
      di += wi[k] * wi[k];
      dn += wo[k] * wo[k];
    }
    di = std::sqrt(di);
    dn = std::sqrt(dn);
    for (int k = 0; k < 3; ++k) {
      wi[k] /= di;
      wo[k] /= dn;
      x[8 + k] = wi[k];
      x[11 + k] = wo[k];
    }
    x[14] = di;
    double v = kY00 * vis_sh[ncoef * i];
    if (sh_degree >= 1)
      v += kY1 * (vis_sh[ncoef * i + 1] * wi[1] + vis_sh[ncoef * i + 2] * wi[2] +
                  vis_sh[ncoef * i + 3] * wi[0]);
    x[15] = std::min(1.0, std::max(0.0, v));
    for (int k = 0; k < 4; ++k) {
      const double fr = (double)(1 << k) * kPi;
      for (int a = 0; a < 3; ++a) {
        x[16 + 6 * k + a] = std::sin(fr * mu[a]);
        x[16 + 6 * k + 3 + a] = std::cos(fr * mu[a]);
      }
    }
    for (int k = 0; k < F; ++k) x[40 + k] = feat[(int64_t)F * i + k];
  }
}

// -------------------------------------------------------------------------------------
// Step 2 -- the MLP.  PAPER.md L100: "share the same MLP but apply separate output heads";
// L347: trunk layers with (Leaky-)ReLU; incident head = optional extra hidden layer(s)
// with the activation, then a ReLU output (1 channel, S12); SSS head = sigmoid output (3).
// params: packed float32, per layer W[out][in] row-major then b[out]; order = trunk layers,
// SSS head, incident hidden layers, incident output.
// mode 0: double reference.  mode 1: bf16-emulating -- every layer INPUT (and the weights,
// already bf16 in the generator) rounded to bf16 RNE, products and sums in double, bias and
// activation in double.  mode 2: fp16-emulating -- the same with binary16
// roundings (round_fp16: RNE, subnormals, finite saturation), the activation precision the
// kernel uses to meet the 1e-2 bound on the unbounded incident output (SURVEY 8(c) measured
// note).  out[i] = (L_SSS r,g,b, L_in).
// -------------------------------------------------------------------------------------
void orc_mlp_forward(int64_t n, const double* x_in, int in_dim, int n_trunk,
                     const int* trunk_width, int n_inc_hidden, const int* inc_hidden_width,
                     int activation, double leaky_slope, const float* params, int mode,
                     double* out) {
  struct Layer {
    const float* W;
    const float* b;
    int o, i;
  };
  std::vector<Layer> trunk, inc;
  Layer sss, inc_out;
  const float* p = params;
  int d = in_dim;
  for (int l = 0; l < n_trunk; ++l) {
    trunk.push_back({p, p + (size_t)trunk_width[l] * d, trunk_width[l], d});
    p += (size_t)trunk_width[l] * d + trunk_width[l];
    d = trunk_width[l];
  }
  sss = {p, p + 3 * (size_t)d, 3, d};
  p += 3 * (size_t)d + 3;
  int di = d;
  for (int l = 0; l < n_inc_hidden; ++l) {
    inc.push_back({p, p + (size_t)inc_hidden_width[l] * di, inc_hidden_width[l], di});
    p += (size_t)inc_hidden_width[l] * di + inc_hidden_width[l];
    di = inc_hidden_width[l];
  }
  inc_out = {p, p + (size_t)di, 1, di};

  auto act = [&](double v) {
    if (activation == ACT_LEAKY_RELU) return v > 0 ? v : leaky_slope * v;
    return v > 0 ? v : 0.0;
  };
  // the rounding of the emulating modes: applied to every weight and to every layer input
  auto rnd = [&](double v) { return mode == 1 ? round_bf16(v) : (mode == 2 ? round_fp16(v) : v); };
  // weights as the tensor cores see them: rounded once (the same value whichever row uses it)
  std::vector<double> Wr((size_t)((p + di + 1) - params));
  for (size_t q = 0; q < Wr.size(); ++q) Wr[q] = rnd((double)params[q]);
  auto linear = [&](const Layer& L, const std::vector<double>& h, std::vector<double>& y) {
    std::vector<double> hr(L.i);
    for (int k = 0; k < L.i; ++k) hr[k] = rnd(h[k]);   // the layer input, rounded
    const double* W = Wr.data() + (L.W - params);
    y.assign(L.o, 0.0);
    for (int o = 0; o < L.o; ++o) {
      double s = 0;
      for (int k = 0; k < L.i; ++k) s += hr[k] * W[(size_t)o * L.i + k];
      y[o] = s + (double)L.b[o];
    }
  };
#pragma omp parallel for schedule(static)
  for (int64_t r = 0; r < n; ++r) {
    std::vector<double> h(x_in + r * in_dim, x_in + (r + 1) * in_dim), y;
    for (const Layer& L : trunk) {
      linear(L, h, y);
      for (double& v : y) v = act(v);
      h.swap(y);
    }
    linear(sss, h, y);
    for (int c = 0; c < 3; ++c) out[4 * r + c] = 1.0 / (1.0 + std::exp(-y[c]));
    std::vector<double> hi = h;
    for (const Layer& L : inc) {
      linear(L, hi, y);
      for (double& v : y) v = act(v);
      hi.swap(y);
    }
    linear(inc_out, hi, y);
    out[4 * r + 3] = y[0] > 0 ? y[0] : 0.0;
  }
}

// -------------------------------------------------------------------------------------
// Step 3 -- EWA projection, Eq. 2: Sigma' = J W Sigma W^T J^T, with
// Sigma = (R_q S)(R_q S)^T from scale s and unit quaternion q (L72).
// CANONICAL FP32 SEQUENCE P1..P10: every operation below is ONE IEEE-754
// binary32 operation (round to nearest even); fmaf is a single rounding; nothing may be
// contracted or re-associated (build with -ffp-contract=off).
//   dot3(a,b)    = fma(a0,b0, fma(a1,b1, a2*b2))
//   dot3p(a,b,c) = fma(a0,b0, fma(a1,b1, fma(a2,b2, c)))
// Outputs per Gaussian: visible (0/1), pix (2), depth, conic (3), radius, rect
// (x0,y0,x1,y1 half-open, in tiles), tiles_touched.  Culled Gaussians get visible = 0,
// tiles_touched = 0 and zeros elsewhere.
// -------------------------------------------------------------------------------------
static inline float dot3(const float* a, const float* b) {
  return fmaf(a[0], b[0], fmaf(a[1], b[1], a[2] * b[2]));
}
static inline float dot3p(const float* a, const float* b, float c) {
  return fmaf(a[0], b[0], fmaf(a[1], b[1], fmaf(a[2], b[2], c)));
}
static inline int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

void orc_project(int64_t n, const float* means, const float* scales, const float* rotations,
                 const OrcCamera* cam, int tile_w, int tile_h, int32_t* visible, float* pix,
                 float* depth, float* conic, float* radius, int32_t* rect, int32_t* touched) {
  const int tiles_x = (cam->width + tile_w - 1) / tile_w;
  const int tiles_y = (cam->height + tile_h - 1) / tile_h;
  const float* R = cam->R;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    visible[i] = 0;
    touched[i] = 0;
    pix[2 * i] = pix[2 * i + 1] = depth[i] = radius[i] = 0.f;
    conic[3 * i] = conic[3 * i + 1] = conic[3 * i + 2] = 0.f;
    rect[4 * i] = rect[4 * i + 1] = rect[4 * i + 2] = rect[4 * i + 3] = 0;
    const float* mu = means + 3 * i;
    // P1: camera transform, near cull
    float p[3];
    for (int k = 0; k < 3; ++k) p[k] = dot3p(R + 3 * k, mu, cam->t[k]);
    const float z = p[2];
    if (!(z > cam->znear)) continue;
    // P2: perspective division, pixel position (pixel k centred at integer k)
    const float u = p[0] / z, w = p[1] / z;
    const float pix_x = fmaf(cam->fx, u, cam->cx), pix_y = fmaf(cam->fy, w, cam->cy);
    // P3: frustum clamp, used by the Jacobian only
    const float lim_x = kFrustumClamp * cam->tan_half_fovx, lim_y = kFrustumClamp * cam->tan_half_fovy;
    const float u_cl = fminf(lim_x, fmaxf(-lim_x, u)), w_cl = fminf(lim_y, fmaxf(-lim_y, w));
    const float x_cl = u_cl * z, y_cl = w_cl * z;
    // P4: Jacobian of the perspective projection
    const float zz = z * z;
    const float j00 = cam->fx / z, j11 = cam->fy / z;
    const float j02 = -((cam->fx * x_cl) / zz), j12 = -((cam->fy * y_cl) / zz);
    // P5: Sigma from the quaternion (r,x,y,z) and the scale
    const float qr = rotations[4 * i], qx = rotations[4 * i + 1], qy = rotations[4 * i + 2],
                qz = rotations[4 * i + 3];
    const float xx = qx * qx, yy = qy * qy, zz2 = qz * qz, xy = qx * qy, xz = qx * qz,
                yz = qy * qz, rx = qr * qx, ry = qr * qy, rz = qr * qz;
    float Rq[9];
    Rq[0] = 1.f - 2.f * (yy + zz2);
    Rq[1] = 2.f * (xy - rz);
    Rq[2] = 2.f * (xz + ry);
    Rq[3] = 2.f * (xy + rz);
    Rq[4] = 1.f - 2.f * (xx + zz2);
    Rq[5] = 2.f * (yz - rx);
    Rq[6] = 2.f * (xz - ry);
    Rq[7] = 2.f * (yz + rx);
    Rq[8] = 1.f - 2.f * (xx + yy);
    float M[9];
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) M[3 * a + b] = Rq[3 * a + b] * scales[3 * i + b];
    float S[9];
    for (int a = 0; a < 3; ++a)
      for (int b = a; b < 3; ++b) S[3 * a + b] = S[3 * b + a] = dot3(M + 3 * a, M + 3 * b);
    // P6: T = J W (2x3), Sigma' = T Sigma T^T, low-pass
    float T0[3], T1[3], g0[3], g1[3];
    for (int k = 0; k < 3; ++k) {
      T0[k] = fmaf(j02, R[6 + k], j00 * R[0 + k]);
      T1[k] = fmaf(j12, R[6 + k], j11 * R[3 + k]);
    }
    for (int k = 0; k < 3; ++k) {
      g0[k] = dot3(S + 3 * k, T0);
      g1[k] = dot3(S + 3 * k, T1);
    }
    const float a = dot3(T0, g0) + kLowPass;
    const float b = dot3(T1, g0);
    const float c = dot3(T1, g1) + kLowPass;
    // P7: determinant, conic = inverse of Sigma'
    const float det = fmaf(a, c, -(b * b));
    if (!(det > 0.f)) continue;
    const float id = 1.f / det;
    const float con_a = c * id, con_b = -(b * id), con_c = a * id;
    // P8: radius from the larger eigenvalue
    const float mid = 0.5f * (a + c);
    const float disc = fmaxf(kDiscFloor, fmaf(mid, mid, -det));
    const float lam = mid + sqrtf(disc);
    const float rad = kRadiusSigma * sqrtf(lam);
    // P8b: non-finite guard (NaN compares false -> culled)
    if (!(fabsf(pix_x) <= 1e9f) || !(fabsf(pix_y) <= 1e9f) || !(rad <= 1e9f)) continue;
    // P9: tile rectangle, half-open, inclusive upper form floor((p+r)/tile)+1
    const int x0 = clampi((int)floorf((pix_x - rad) / (float)tile_w), 0, tiles_x);
    const int x1 = clampi((int)floorf((pix_x + rad) / (float)tile_w) + 1, 0, tiles_x);
    const int y0 = clampi((int)floorf((pix_y - rad) / (float)tile_h), 0, tiles_y);
    const int y1 = clampi((int)floorf((pix_y + rad) / (float)tile_h) + 1, 0, tiles_y);
    const int cnt = (x1 - x0) * (y1 - y0);
    if (cnt <= 0) continue;
    visible[i] = 1;
    touched[i] = cnt;
    pix[2 * i] = pix_x;
    pix[2 * i + 1] = pix_y;
    depth[i] = z;  // P10: key depth bits = bit pattern of z (z > 0)
    conic[3 * i] = con_a;
    conic[3 * i + 1] = con_b;
    conic[3 * i + 2] = con_c;
    radius[i] = rad;
    rect[4 * i] = x0;
    rect[4 * i + 1] = y0;
    rect[4 * i + 2] = x1;
    rect[4 * i + 3] = y1;
  }
}

// The same projection written directly from Eq. 2 in double with 3x3 matrix products
// (no canonical ordering); tests assert agreement with orc_project to ~1e-5 relative, so
// that the canonical text itself is checked.  Outputs cov2d (a,b,c incl. low-pass), pix, depth.
void orc_project_f64(int64_t n, const float* means, const float* scales, const float* rotations,
                     const OrcCamera* cam, double* cov2d, double* pix, double* depth) {
  for (int64_t i = 0; i < n; ++i) {
    double R[9], t[3];
    for (int k = 0; k < 9; ++k) R[k] = cam->R[k];
    for (int k = 0; k < 3; ++k) t[k] = cam->t[k];
    double p[3];
    for (int k = 0; k < 3; ++k)
      p[k] = R[3 * k] * means[3 * i] + R[3 * k + 1] * means[3 * i + 1] + R[3 * k + 2] * means[3 * i + 2] + t[k];
    depth[i] = p[2];
    const double u = p[0] / p[2], w = p[1] / p[2];
    pix[2 * i] = cam->fx * u + cam->cx;
    pix[2 * i + 1] = cam->fy * w + cam->cy;
    const double lx = 1.3 * cam->tan_half_fovx, ly = 1.3 * cam->tan_half_fovy;
    const double xc = std::min(lx, std::max(-lx, u)) * p[2], yc = std::min(ly, std::max(-ly, w)) * p[2];
    const double J[6] = {cam->fx / p[2], 0, -cam->fx * xc / (p[2] * p[2]),
                         0, cam->fy / p[2], -cam->fy * yc / (p[2] * p[2])};
    const double r = rotations[4 * i], x = rotations[4 * i + 1], y = rotations[4 * i + 2], z = rotations[4 * i + 3];
    const double Rq[9] = {1 - 2 * (y * y + z * z), 2 * (x * y - r * z), 2 * (x * z + r * y),
                          2 * (x * y + r * z), 1 - 2 * (x * x + z * z), 2 * (y * z - r * x),
                          2 * (x * z - r * y), 2 * (y * z + r * x), 1 - 2 * (x * x + y * y)};
    double M[9], Sg[9], T[6], TS[6];
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) M[3 * a + b] = Rq[3 * a + b] * scales[3 * i + b];
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) {
        double s = 0;
        for (int k = 0; k < 3; ++k) s += M[3 * a + k] * M[3 * b + k];
        Sg[3 * a + b] = s;
      }
    for (int a = 0; a < 2; ++a)
      for (int b = 0; b < 3; ++b) {
        double s = 0;
        for (int k = 0; k < 3; ++k) s += J[3 * a + k] * R[3 * k + b];
        T[3 * a + b] = s;
      }
    for (int a = 0; a < 2; ++a)
      for (int b = 0; b < 3; ++b) {
        double s = 0;
        for (int k = 0; k < 3; ++k) s += T[3 * a + k] * Sg[3 * k + b];
        TS[3 * a + b] = s;
      }
    double c2[4];
    for (int a = 0; a < 2; ++a)
      for (int b = 0; b < 2; ++b) {
        double s = 0;
        for (int k = 0; k < 3; ++k) s += TS[3 * a + k] * T[3 * b + k];
        c2[2 * a + b] = s;
      }
    cov2d[3 * i] = c2[0] + 0.3;
    cov2d[3 * i + 1] = c2[1];
    cov2d[3 * i + 2] = c2[3] + 0.3;
  }
}

// -------------------------------------------------------------------------------------
// Step 4 -- keys, sort, tile ranges ("efficiently designed splatting
// technique", L68 "layered sequenced Gaussians"; design per SURVEY 8(c) step 4 / S6).
// For Gaussian index ascending, tile y then x ascending: key = (y*tiles_x + x) << 32 |
// bits(depth), value = Gaussian index.  std::stable_sort by key (ties -> ascending index).
// ranges[t] = [lower_bound(t<<32), lower_bound((t+1)<<32)).
// Call with keys == nullptr to get the instance count only.
// -------------------------------------------------------------------------------------
int64_t orc_build_lists(int64_t n, const int32_t* rect, const float* depth, const int32_t* touched,
                        int tiles_x, int tiles_y, uint64_t* keys, uint32_t* vals, uint32_t* ranges) {
  int64_t total = 0;
  for (int64_t i = 0; i < n; ++i) total += touched[i];
  if (!keys) return total;
  std::vector<std::pair<uint64_t, uint32_t>> kv;
  kv.reserve(total);
  for (int64_t i = 0; i < n; ++i) {
    if (!touched[i]) continue;
    uint32_t dbits;
    std::memcpy(&dbits, depth + i, 4);
    for (int y = rect[4 * i + 1]; y < rect[4 * i + 3]; ++y)
      for (int x = rect[4 * i]; x < rect[4 * i + 2]; ++x)
        kv.push_back({((uint64_t)(y * tiles_x + x) << 32) | dbits, (uint32_t)i});
  }
  std::stable_sort(kv.begin(), kv.end(),
                   [](const auto& a, const auto& b) { return a.first < b.first; });
  for (int64_t j = 0; j < total; ++j) {
    keys[j] = kv[j].first;
    vals[j] = kv[j].second;
  }
  const int tiles = tiles_x * tiles_y;
  for (int t = 0; t < tiles; ++t) {
    auto lb = [&](uint64_t k) {
      return (uint32_t)(std::lower_bound(keys, keys + total, k) - keys);
    };
    ranges[2 * t] = lb((uint64_t)t << 32);
    ranges[2 * t + 1] = lb((uint64_t)(t + 1) << 32);
  }
  return total;
}

// -------------------------------------------------------------------------------------
// Step 5 / 7 -- front-to-back alpha compositing, Eq. 3:
//   C = sum_i ( prod_{j<i} (1 - alpha_j) ) alpha_i c_i,
//   alpha = opacity x 2-D Gaussian falloff of Sigma' at the pixel (L72),
// applied to every property channel (L55: "accumulate and rasterize each property on the
// image plane in a deferred shading pipeline").  Rules (S3, S4): d = p - pix_i;
// power = -1/2 (A dx^2 + C dy^2) - B dx dy; skip if power > 0; alpha = min(0.99, o exp(power));
// skip if alpha < 1/255; T' = T (1 - alpha); if T' < 1e-4 stop (this Gaussian is NOT
// blended); acc_c += T alpha ch_c; T = T'.
// G-buffer pixel (16 doubles, un-normalised accumulations):
//   [0] depth [1-3] normal [4-6] base [7] rough [8] metal [9] sss [10-12] L_SSS [13] L_in
//   [14] A = sum of weights [15] T_final.
// ch = per-Gaussian channel values [n][14] in the order of G-buffer channels 0..13.
// order/ranges: tiled mode  -> order = sorted values list, ranges = per-tile [begin,end);
//               brute mode  -> ranges == nullptr, order = ALL visible Gaussians sorted by
//                              (depth bits, index), n_order entries; no tiles involved.
// unstable[p] != 0 if any skip/stop decision at p sits within the fp32 evaluation error of
// its threshold (S7): such pixels may legitimately differ between correct implementations.
// The value says which rule flagged the pixel: bit 0 = power within rounding of 0 (skip vs
// blend at alpha = o), bit 1 = alpha within rounding of 1/255, bit 2 = T' within 1e-3 relative
// of 1e-4; bits 4-7 = number of alpha-threshold decisions flagged at the pixel (saturating at 15).
// counters: [0] P_eval (list entries visited, up to and including the stopping entry),
//           [1] P_blend (blended entries), [2] unstable pixels, [3] / [4] / [5] pixels flagged
//           by the power / alpha / T rule.
// contrib[g] = 1 if Gaussian g was blended at >= 1 pixel (may be nullptr).
// -------------------------------------------------------------------------------------
void orc_composite(int width, int height, int tile_w, int tile_h, const float* pix,
                   const float* conic, const float* opacities, const double* ch,
                   const uint32_t* order, int64_t n_order, const uint32_t* ranges,
                   double* gbuf, uint8_t* unstable, int64_t* counters, uint8_t* contrib) {
  const int tiles_x = (width + tile_w - 1) / tile_w;
  int64_t p_eval = 0, p_blend = 0, n_unstable = 0, n_rule_p = 0, n_rule_a = 0, n_rule_t = 0;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : p_eval, p_blend, n_unstable, n_rule_p, n_rule_a, n_rule_t)
  for (int py = 0; py < height; ++py) {
    for (int px = 0; px < width; ++px) {
      int64_t begin = 0, end = n_order;
      if (ranges) {
        const int t = (py / tile_h) * tiles_x + (px / tile_w);
        begin = ranges[2 * t];
        end = ranges[2 * t + 1];
      }
      double acc[14] = {0};
      double T = 1.0, A = 0.0;
      unsigned flags = 0, n_alpha_flags = 0;  // which rule flagged the pixel (diagnostic only)
      for (int64_t j = begin; j < end; ++j) {
        const uint32_t g = order[j];
        ++p_eval;
        const double dx = (double)px - (double)pix[2 * g], dy = (double)py - (double)pix[2 * g + 1];
        const double ca = conic[3 * g], cb = conic[3 * g + 1], cc = conic[3 * g + 2];
        const double power = -0.5 * (ca * dx * dx + cc * dy * dy) - cb * dx * dy;
        // magnitude of the terms: bounds the fp32 evaluation error of `power`
        const double mag = 0.5 * (std::fabs(ca) * dx * dx + std::fabs(cc) * dy * dy) + std::fabs(cb * dx * dy);
        const double perr = 1e-5 + 16.0 * 5.96e-8 * mag;
        if (std::fabs(power) < perr && power > -perr) {
          // power within rounding of 0: skip-vs-blend is ambiguous only if alpha matters
          if ((double)opacities[g] >= kAlphaMin) flags |= 1u;
        }
        if (power > 0.0) continue;
        const double araw = (double)opacities[g] * std::exp(power);
        const double alpha = std::min(kAlphaMax, araw);
        if (std::fabs(alpha - kAlphaMin) <= perr * kAlphaMin) { flags |= 2u; ++n_alpha_flags; }
        if (alpha < kAlphaMin) continue;
        const double Tn = T * (1.0 - alpha);
        if (std::fabs(Tn - kTMin) <= 1e-3 * kTMin) flags |= 4u;
        if (Tn < kTMin) break;
        const double w = T * alpha;
        for (int c = 0; c < 14; ++c) acc[c] += w * ch[14 * (int64_t)g + c];
        A += w;
        T = Tn;
        ++p_blend;
        if (contrib) contrib[g] = 1;  // benign race: every writer stores 1
      }
      double* o = gbuf + ((int64_t)py * width + px) * kGbufChannels;
      for (int c = 0; c < 14; ++c) o[c] = acc[c];
      o[14] = A;
      o[15] = T;
      unstable[(int64_t)py * width + px] = (uint8_t)(flags | ((n_alpha_flags > 15u ? 15u : n_alpha_flags) << 4));
      n_unstable += flags ? 1 : 0;
      n_rule_p += (flags & 1u) ? 1 : 0;
      n_rule_a += (flags & 2u) ? 1 : 0;
      n_rule_t += (flags & 4u) ? 1 : 0;
    }
  }
  counters[0] = p_eval;
  counters[1] = p_blend;
  counters[2] = n_unstable;
  counters[3] = n_rule_p;
  counters[4] = n_rule_a;
  counters[5] = n_rule_t;
}

// -------------------------------------------------------------------------------------
// Tight tile lists ("efficiently designed splatting technique").  The
// canonical list holds every (tile, Gaussian) pair of the Gaussian's tile rectangle; a valid tight
// list is a sub-sequence of it that still contains every pair with alpha >= 1/255 at SOME pixel of
// the tile (only those can ever be blended, whatever the transmittance).  This function computes that
// minimal set from the definition: for entry j of the sorted list, lying in tile t, hit[j] = 1 iff
//   exists pixel p of tile t (inside the image):  power(p) <= 0  and  min(0.99, o exp(power(p))) >= 1/255,
// with power as in orc_composite.  Brute force over the pixels of the tile.
// -------------------------------------------------------------------------------------
void orc_tile_hits(int width, int height, int tile_w, int tile_h, const float* pix, const float* conic,
                   const float* opacities, const uint32_t* order, const uint32_t* ranges, int tiles_x,
                   int tiles_y, uint8_t* hit) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int t = 0; t < tiles_x * tiles_y; ++t) {
    const int px0 = (t % tiles_x) * tile_w, py0 = (t / tiles_x) * tile_h;
    const int px1 = std::min(px0 + tile_w, width), py1 = std::min(py0 + tile_h, height);
    for (uint32_t j = ranges[2 * t]; j < ranges[2 * t + 1]; ++j) {
      const uint32_t g = order[j];
      const double ca = conic[3 * g], cb = conic[3 * g + 1], cc = conic[3 * g + 2];
      uint8_t h = 0;
      for (int py = py0; py < py1 && !h; ++py)
        for (int px = px0; px < px1; ++px) {
          const double dx = (double)px - (double)pix[2 * g], dy = (double)py - (double)pix[2 * g + 1];
          const double power = -0.5 * (ca * dx * dx + cc * dy * dy) - cb * dx * dy;
          if (power > 0.0) continue;
          if (std::min(kAlphaMax, (double)opacities[g] * std::exp(power)) >= kAlphaMin) {
            h = 1;
            break;
          }
        }
      hit[j] = h;
    }
  }
}

// -------------------------------------------------------------------------------------
// Step 6 -- per-pixel deferred shading.  PAPER.md L114: "evaluate the BRDF model in image
// space after the rasterization ... The image space surface position is projected back to
// the 3D space"; L76-80 Eq. 4 (Disney/Cook-Torrance: f_diffuse = (1-m)/pi b,
// f_specular = D F G / ((w_o.n)(w_i.n))); L104-106 Eq. 7:
//   L_out = sss L_SSS + (1 - sss)(f_specular + f_diffuse) L_in (n . w_in).
// Readings: S10 normalise the accumulated channels by coverage A, shade, re-apply A and the
// background; S8 the standard Cook-Torrance normalisation (the 4 that Eq. 4 omits), GGX D
// with alpha_r = r^2 (floored at 1e-3), Schlick F with F0 = 0.04(1-m) + b m, Smith-Schlick
// visibility with k = alpha_r/2; S16 point light without explicit 1/d^2, RGB intensity;
// S17 linear output.  D uses the cancellation-free form
//   D = a^2 / (pi (a^2 nh^2 + |n x h|^2)^2),  since 1 - nh^2 = |n x h|^2 for unit n, h  (S9).
// AOVs (L320: "Specular and diffuse illumination ... before multiplication with the base
// color"): diffuse = (1-sss)(1-m)/pi L_in nl (replicated to 3 channels),
//          specular = (1-sss) f_spec L_in nl; both 0 where A < 1e-6.
// Template on the arithmetic type: double = the oracle; float = the plain-fp32 evaluation
// of the same text used only to calibrate tolerances at ill-conditioned highlights (S9).
// -------------------------------------------------------------------------------------
}  // extern "C"

template <typename real>
static void shade_impl(int width, int height, const OrcCamera* cam, const float* light_pos,
                       const float* light_intensity, const double* gbuf, real* rgb, real* aov_d,
                       real* aov_s) {
  real pc[3];
  for (int k = 0; k < 3; ++k)
    pc[k] = -((real)cam->R[0 + k] * (real)cam->t[0] + (real)cam->R[3 + k] * (real)cam->t[1] +
              (real)cam->R[6 + k] * (real)cam->t[2]);
  const real pi = (real)kPi;
#pragma omp parallel for schedule(static) if (height > 4)
  for (int py = 0; py < height; ++py)
    for (int px = 0; px < width; ++px) {
      const int64_t pidx = (int64_t)py * width + px;
      real g[16];
      for (int c = 0; c < 16; ++c) g[c] = (real)gbuf[pidx * 16 + c];
      real* o = rgb + 3 * pidx;
      real dif[3] = {0, 0, 0}, spc[3] = {0, 0, 0};
      const real A = g[14];
      if (A < (real)1e-6) {
        for (int c = 0; c < 3; ++c) o[c] = (real)cam->bg[c];
      } else {
        real q[14];
        for (int c = 0; c < 14; ++c) q[c] = g[c] / A;
        const real zb = q[0], rough = q[7], metal = q[8], sss = q[9], lin = q[13];
        // back-projection of the pixel at depth zb: x_cam = ((px-cx)/fx zb, (py-cy)/fy zb, zb)
        const real xc[3] = {((real)px - (real)cam->cx) / (real)cam->fx * zb,
                            ((real)py - (real)cam->cy) / (real)cam->fy * zb, zb};
        real xw[3];
        for (int k = 0; k < 3; ++k)
          xw[k] = (real)cam->R[0 + k] * (xc[0] - (real)cam->t[0]) +
                  (real)cam->R[3 + k] * (xc[1] - (real)cam->t[1]) +
                  (real)cam->R[6 + k] * (xc[2] - (real)cam->t[2]);
        real l[3], v[3], ll = 0, lv = 0;
        for (int k = 0; k < 3; ++k) {
          l[k] = (real)light_pos[k] - xw[k];
          v[k] = pc[k] - xw[k];
          ll += l[k] * l[k];
          lv += v[k] * v[k];
        }
        ll = std::sqrt(ll);
        lv = std::sqrt(lv);
        for (int k = 0; k < 3; ++k) {
          l[k] /= ll;
          v[k] /= lv;
        }
        real nn = std::sqrt(q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
        real brdf_l[3] = {0, 0, 0};  // (f_spec + f_diff) L_in nl
        if (nn >= (real)1e-8) {
          const real n[3] = {q[1] / nn, q[2] / nn, q[3] / nn};
          real h[3] = {l[0] + v[0], l[1] + v[1], l[2] + v[2]};
          const real hl = std::sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
          if (hl >= (real)1e-8) {
            for (int k = 0; k < 3; ++k) h[k] /= hl;
          } else {
            for (int k = 0; k < 3; ++k) h[k] = n[k];
          }
          const real nl = std::max((real)0, n[0] * l[0] + n[1] * l[1] + n[2] * l[2]);
          const real nv = std::max((real)1e-4, n[0] * v[0] + n[1] * v[1] + n[2] * v[2]);
          const real nh = std::min((real)1, std::max((real)0, n[0] * h[0] + n[1] * h[1] + n[2] * h[2]));
          const real vh = std::min((real)1, std::max((real)0, v[0] * h[0] + v[1] * h[1] + v[2] * h[2]));
          const real ar = std::max((real)1e-3, rough * rough);
          const real a2 = ar * ar;
          const real cx = n[1] * h[2] - n[2] * h[1], cy = n[2] * h[0] - n[0] * h[2],
                     cz = n[0] * h[1] - n[1] * h[0];
          const real s2 = cx * cx + cy * cy + cz * cz;
          // >= a2 >= 1e-6 for any unit n, h with nh in [0,1]; the floor only catches n = -h exactly
          // (nh clamped to 0 and |n x h| = 0), where D would be a2 / 0
          const real dd = std::max((real)1e-12, a2 * nh * nh + s2);
          const real D = a2 / (pi * dd * dd);
          const real k = ar * (real)0.5;
          const real V = (real)1 / ((real)4 * (nl * ((real)1 - k) + k) * (nv * ((real)1 - k) + k));
          const real om = (real)1 - vh;
          const real om5 = om * om * om * om * om;
          for (int c = 0; c < 3; ++c) {
            const real F0 = (real)0.04 * ((real)1 - metal) + q[4 + c] * metal;
            const real F = F0 + ((real)1 - F0) * om5;
            const real fs = D * F * V;
            const real fd = ((real)1 - metal) * q[4 + c] / pi;
            brdf_l[c] = (fs + fd) * lin * nl;
            spc[c] = ((real)1 - sss) * fs * lin * nl;
            dif[c] = ((real)1 - sss) * ((real)1 - metal) / pi * lin * nl;
          }
        }
        for (int c = 0; c < 3; ++c) {
          const real lout = sss * q[10 + c] + ((real)1 - sss) * brdf_l[c];
          o[c] = (real)light_intensity[c] * A * lout + ((real)1 - A) * (real)cam->bg[c];
        }
      }
      if (aov_d)
        for (int c = 0; c < 3; ++c) aov_d[3 * pidx + c] = dif[c];
      if (aov_s)
        for (int c = 0; c < 3; ++c) aov_s[3 * pidx + c] = spc[c];
    }
}

extern "C" {

void orc_shade(int width, int height, const OrcCamera* cam, const float* light_pos,
               const float* light_intensity, const double* gbuf, double* rgb, double* aov_d,
               double* aov_s) {
  shade_impl<double>(width, height, cam, light_pos, light_intensity, gbuf, rgb, aov_d, aov_s);
}
void orc_shade_f32(int width, int height, const OrcCamera* cam, const float* light_pos,
                   const float* light_intensity, const double* gbuf, float* rgb, float* aov_d,
                   float* aov_s) {
  shade_impl<float>(width, height, cam, light_pos, light_intensity, gbuf, rgb, aov_d, aov_s);
}

}  // extern "C"

extern "C" {

// ---------------------------------------------------------------------------------------------
// Ray-traced per-Gaussian visibility and its SH fit ("we trace
// rays using a BVH to quickly estimate the visibility for each Gaussian and learn this as a per
// Gaussian SH visibility term v"; L81: "efficient ray-tracing for 3D GS").  The paper gives no
// formula; the reading is the one of its reference [10]: along the ray
// x(t) = mu_i + (t_min + t) w, t >= 0, every other Gaussian j acts at the point of its largest
// response, with the opacity rule of the rasteriser (Eq. 3: alpha = o * falloff, capped,
// thresholded), and the transmittances multiply:
//   m2_ij  = min_{t >= 0} (x(t) - mu_j)^T Sigma_j^-1 (x(t) - mu_j)
//   a_ij   = min(0.99, o_j exp(-m2_ij / 2)), counted iff a_ij >= 1/255
//   V_i(w) = prod_{j != i} (1 - a_ij), set to 0 below 1e-4 (the product is order independent)
//   c_i,lm = sum_k weight_k V_i(w_k) Y_lm(w_k)      (quadrature of the SH projection, degree <= 1,
//            real basis and order of the render path: Y00, Y1-1 ~ y, Y10 ~ z, Y11 ~ x)
// Brute force over all pairs, in double; no BVH here: the tree only prunes pairs whose a_ij is
// below the threshold.  `unstable` counts, per ray, the pairs whose a_ij lies within 1e-4 relative
// of 1/255 plus one if the product lies within 1e-2 relative of 1e-4 (a float evaluation may
// decide these the other way).
void orc_bake_visibility(int64_t n, const float* means, const float* scales, const float* rotations,
                         const float* opacities, int n_dirs, const float* dirs, const float* weights,
                         float t_min, int sh_degree, int positions, int64_t n_rows, const int64_t* rows,
                         double* sh_out, double* vis_out, int32_t* unstable) {
  // positions != 0: `dirs` holds K points p_k (the OLAT lights of L110, "the position of the light
  // source is known"): the ray of Gaussian i runs from mu_i towards p_k and ends there,
  // w = (p_k - mu_i) / d, t in [0, d - t_min]; nothing occludes if d <= t_min.
  // rows: the Gaussians whose rays are traced (all n if NULL); outputs are indexed by position in rows
  const int nc = (sh_degree + 1) * (sh_degree + 1);
  std::vector<double> Sinv((size_t)n * 9);
  for (int64_t j = 0; j < n; ++j) {
    const double qr = rotations[4 * j], qx = rotations[4 * j + 1], qy = rotations[4 * j + 2],
                 qz = rotations[4 * j + 3];
    double R[9];
    R[0] = 1 - 2 * (qy * qy + qz * qz); R[1] = 2 * (qx * qy - qr * qz); R[2] = 2 * (qx * qz + qr * qy);
    R[3] = 2 * (qx * qy + qr * qz); R[4] = 1 - 2 * (qx * qx + qz * qz); R[5] = 2 * (qy * qz - qr * qx);
    R[6] = 2 * (qx * qz - qr * qy); R[7] = 2 * (qy * qz + qr * qx); R[8] = 1 - 2 * (qx * qx + qy * qy);
    // Sigma = R S^2 R^T  =>  Sigma^-1 = R S^-2 R^T
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) {
        double s = 0;
        for (int k = 0; k < 3; ++k) {
          const double sk = scales[3 * j + k];
          s += R[3 * a + k] * R[3 * b + k] / (sk * sk);
        }
        Sinv[9 * j + 3 * a + b] = s;
      }
  }
  if (!rows) n_rows = n;
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t r = 0; r < n_rows; ++r) {
    const int64_t i = rows ? rows[r] : r;
    double c[4] = {0, 0, 0, 0};
    for (int k = 0; k < n_dirs; ++k) {
      double w[3] = {dirs[3 * k], dirs[3 * k + 1], dirs[3 * k + 2]};
      double t_max = INFINITY;
      if (positions) {
        double d2 = 0;
        for (int a = 0; a < 3; ++a) { w[a] -= (double)means[3 * i + a]; d2 += w[a] * w[a]; }
        const double d = std::sqrt(d2);
        for (int a = 0; a < 3; ++a) w[a] = d > 0 ? w[a] / d : 0.0;
        t_max = d - (double)t_min;
      }
      double o[3];
      for (int a = 0; a < 3; ++a) o[a] = (double)means[3 * i + a] + (double)t_min * w[a];
      double T = 1.0;
      int flips = 0;
      for (int64_t j = 0; j < n; ++j) {
        if (j == i || !(t_max > 0)) continue;
        const double* S = &Sinv[9 * j];
        double d[3], Sw[3], Sd[3];
        for (int a = 0; a < 3; ++a) d[a] = o[a] - (double)means[3 * j + a];
        for (int a = 0; a < 3; ++a) {
          Sw[a] = S[3 * a] * w[0] + S[3 * a + 1] * w[1] + S[3 * a + 2] * w[2];
          Sd[a] = S[3 * a] * d[0] + S[3 * a + 1] * d[1] + S[3 * a + 2] * d[2];
        }
        const double ww = w[0] * Sw[0] + w[1] * Sw[1] + w[2] * Sw[2];
        const double wd = w[0] * Sd[0] + w[1] * Sd[1] + w[2] * Sd[2];
        double t = -wd / ww;  // minimiser of the quadratic along the line
        if (t < 0) t = 0;
        if (t > t_max) t = t_max;
        double e[3], Se[3];
        for (int a = 0; a < 3; ++a) e[a] = d[a] + t * w[a];
        for (int a = 0; a < 3; ++a) Se[a] = S[3 * a] * e[0] + S[3 * a + 1] * e[1] + S[3 * a + 2] * e[2];
        const double m2 = e[0] * Se[0] + e[1] * Se[1] + e[2] * Se[2];
        double a_ij = (double)opacities[j] * std::exp(-0.5 * m2);
        if (std::fabs(a_ij * 255.0 - 1.0) < 1e-4) ++flips;
        if (a_ij < 1.0 / 255.0) continue;
        if (a_ij > 0.99) a_ij = 0.99;
        T *= 1.0 - a_ij;
      }
      if (std::fabs(T * 1e4 - 1.0) < 1e-2) ++flips;
      const double V = T >= 1e-4 ? T : 0.0;
      if (vis_out) vis_out[r * n_dirs + k] = V;
      if (unstable) unstable[r * n_dirs + k] = flips;
      const double wk = weights[k];
      c[0] += wk * V * 0.2820948;
      if (nc == 4) {
        c[1] += wk * V * 0.4886025 * w[1];
        c[2] += wk * V * 0.4886025 * w[2];
        c[3] += wk * V * 0.4886025 * w[0];
      }
    }
    for (int m = 0; m < nc; ++m) sh_out[r * nc + m] = c[m];
  }
}

}  // extern "C"

// Backward pass of hot-path steps a8 (deferred shading), a7 (compositing), a2 (the MLP), a3 (projection) and a1
// (the MLP's input assembly)
// ("optimize all parameters jointly via raytraced differentiable rendering",
// L112, L343-349: the losses are functions of the rendered image and of the rasterised property images).
//
// For one camera and its lights, with G_l = dL / d rgb_l given by the caller (L = sum_l <G_l, rgb_l>):
//   shade_backward_kernel      per (light, pixel): dL / d gbuffer_l[p][0..15]           (Eq. 4, Eq. 7)
//   composite_backward_kernel  per tile, walking its list back to front: dL / d (opacity, 2-D mean, conic,
//                              depth, normal, base colour, roughness, metalness, sss) per Gaussian and
//                              dL / d (L_SSS, L_in) per (Gaussian, light)                        (Eq. 3)
//   project_backward_kernel    dL / d (mean, scale, rotation) from dL / d (2-D mean, conic, depth)    (Eq. 2)
//   mlp_backward_tc_kernel     dL / d Theta (weights and biases of every layer) on the tensor cores (Eq. 6):
//                              binary16 operands, fp32 accumulation, the forward re-evaluated per row tile
//   mlp_backward_kernel        the same in fp32 on the CUDA cores (SSSGS_BACKWARD_FP32; MLPs with incident-head
//                              hidden layers or more than 4 trunk layers)
// The discontinuous decisions of the forward pass (alpha >= 1/255, power <= 0, the T' < 1e-4 stop, the 0.99
// clamp, the ReLUs) are constants of the differentiation.  Shading and compositing backward are fp32.
// Per-Gaussian sums are formed with float atomics: results are reproducible to rounding, not bit for bit.
#include <cuda_fp16.h>

#include <cstdio>
#include <cstring>

#include "internal.cuh"

namespace sssgs {

namespace {

constexpr float kPiF = 3.14159265358979323846f;

__device__ __forceinline__ float dot3f(const float* a, const float* b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
__device__ __forceinline__ void cross3f(const float* a, const float* b, float* c) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}
// x = y / |y|: adjoint of y given the adjoint of x
__device__ __forceinline__ void normalize_bwd(const float* x, float inv_len, const float* dx, float* dy) {
  const float p = dot3f(x, dx);
  for (int k = 0; k < 3; ++k) dy[k] = (dx[k] - x[k] * p) * inv_len;
}

// ---- a8 backward: one thread per (light, pixel) -------------------------------------------------------
__global__ void __launch_bounds__(256)
shade_backward_kernel(CamParams cam, LightBatch lights, int n_lights, int64_t npix,
                      const float* __restrict__ gbuf, const float* __restrict__ grad_rgb,
                      const float* __restrict__ grad_gbuf_in, float* __restrict__ grad_gbuf) {
  const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (i >= npix * n_lights) return;
  const int l_idx = (int)(i / npix);
  const int64_t p = i % npix;
  const int px = (int)(p % cam.width), py = (int)(p / cam.width);
  const float4* gp = reinterpret_cast<const float4*>(gbuf + i * 16);
  float G[16];
  for (int q = 0; q < 4; ++q) {
    const float4 v = gp[q];
    G[4 * q] = v.x; G[4 * q + 1] = v.y; G[4 * q + 2] = v.z; G[4 * q + 3] = v.w;
  }
  float dG[16];
  for (int c = 0; c < 16; ++c) dG[c] = 0.f;
  const float A = G[14];
  const float g[3] = {grad_rgb[i * 3], grad_rgb[i * 3 + 1], grad_rgb[i * 3 + 2]};
  if (A >= 1e-6f) {
    const LightParams& lt = lights.l[l_idx];
    const float iA = 1.f / A;
    float q[14];
    for (int c = 0; c < 14; ++c) q[c] = G[c] * iA;
    const float z = q[0], rough = q[7], metal = q[8], sss = q[9], lin = q[13];
    const float ax = ((float)px - cam.cx) / cam.fx, ay = ((float)py - cam.cy) / cam.fy;
    const float xc[3] = {ax * z - cam.t[0], ay * z - cam.t[1], z - cam.t[2]};
    float xw[3], lv[3], vv[3];
    for (int k = 0; k < 3; ++k) {
      xw[k] = cam.R[0 + k] * xc[0] + cam.R[3 + k] * xc[1] + cam.R[6 + k] * xc[2];
      lv[k] = lt.pos[k] - xw[k];
      vv[k] = cam.pos[k] - xw[k];
    }
    const float il = 1.f / sqrtf(dot3f(lv, lv)), iv = 1.f / sqrtf(dot3f(vv, vv));
    float l[3], v[3];
    for (int k = 0; k < 3; ++k) { l[k] = lv[k] * il; v[k] = vv[k] * iv; }
    const float nraw[3] = {q[1], q[2], q[3]};
    const float nn = sqrtf(dot3f(nraw, nraw));
    const bool has_n = nn >= 1e-8f;
    float d_q[14];
    for (int c = 0; c < 14; ++c) d_q[c] = 0.f;
    // rgb_c = I_c A lout_c + (1 - A) bg_c,  lout_c = s Ls_c + (1 - s) brdf_c
    float brdf[3] = {0.f, 0.f, 0.f};
    float n[3] = {0.f, 0.f, 0.f}, h[3] = {0.f, 0.f, 0.f}, hs[3], ihl = 0.f;
    bool has_h = false;
    float nl = 0.f, nv = 0.f, nh = 0.f, vh = 0.f, ndl = 0.f, ndv = 0.f, ndh = 0.f, vdh = 0.f;
    float ar = 0.f, a2 = 0.f, s2 = 0.f, dd = 0.f, Dg = 0.f, kk = 0.f, Va = 0.f, Vb = 0.f, Vg = 0.f, om = 0.f, om5 = 0.f;
    float cxh[3] = {0.f, 0.f, 0.f}, F0[3], F[3], B[3] = {0.f, 0.f, 0.f};
    if (has_n) {
      for (int k = 0; k < 3; ++k) { n[k] = nraw[k] / nn; hs[k] = l[k] + v[k]; }
      const float hl = sqrtf(dot3f(hs, hs));
      has_h = hl >= 1e-8f;
      ihl = has_h ? 1.f / hl : 0.f;
      for (int k = 0; k < 3; ++k) h[k] = has_h ? hs[k] * ihl : n[k];
      ndl = dot3f(n, l); ndv = dot3f(n, v); ndh = dot3f(n, h); vdh = dot3f(v, h);
      nl = fmaxf(0.f, ndl); nv = fmaxf(1e-4f, ndv); nh = fminf(1.f, fmaxf(0.f, ndh)); vh = fminf(1.f, fmaxf(0.f, vdh));
      ar = fmaxf(1e-3f, rough * rough);
      a2 = ar * ar;
      cross3f(n, h, cxh);
      s2 = dot3f(cxh, cxh);
      dd = fmaxf(1e-12f, a2 * nh * nh + s2);
      Dg = a2 / (kPiF * dd * dd);
      kk = 0.5f * ar;
      Va = nl * (1.f - kk) + kk; Vb = nv * (1.f - kk) + kk;
      Vg = 1.f / (4.f * Va * Vb);
      om = 1.f - vh;
      om5 = om * om * om * om * om;
      for (int c = 0; c < 3; ++c) {
        F0[c] = 0.04f * (1.f - metal) + q[4 + c] * metal;
        F[c] = F0[c] + (1.f - F0[c]) * om5;
        B[c] = Dg * Vg * F[c] + (1.f - metal) * q[4 + c] / kPiF;
        brdf[c] = B[c] * lin * nl;
      }
    }
    float dA = 0.f, d_lout[3], d_brdf[3];
    for (int c = 0; c < 3; ++c) {
      const float lout = sss * q[10 + c] + (1.f - sss) * brdf[c];
      d_lout[c] = g[c] * lt.intensity[c] * A;
      dA += g[c] * (lt.intensity[c] * lout - cam.bg[c]);
      d_q[9] += d_lout[c] * (q[10 + c] - brdf[c]);
      d_q[10 + c] = d_lout[c] * sss;
      d_brdf[c] = d_lout[c] * (1.f - sss);
    }
    if (has_n) {
      float d_B[3], d_nl = 0.f, d_F[3], d_D = 0.f, d_V = 0.f, d_om5 = 0.f, sBF = 0.f;
      for (int c = 0; c < 3; ++c) {
        d_B[c] = d_brdf[c] * lin * nl;
        d_q[13] += d_brdf[c] * B[c] * nl;
        d_nl += d_brdf[c] * B[c] * lin;
        d_q[8] += -d_B[c] * q[4 + c] / kPiF;          // fd = (1 - m) b / pi
        d_q[4 + c] += d_B[c] * (1.f - metal) / kPiF;
        sBF += d_B[c] * F[c];
        d_F[c] = d_B[c] * Dg * Vg;
        const float d_F0 = d_F[c] * (1.f - om5);
        d_om5 += d_F[c] * (1.f - F0[c]);
        d_q[8] += d_F0 * (q[4 + c] - 0.04f);          // F0 = 0.04 (1 - m) + b m
        d_q[4 + c] += d_F0 * metal;
      }
      d_D = Vg * sBF;
      d_V = Dg * sBF;
      float d_vh = (vdh > 0.f && vdh < 1.f) ? -5.f * om * om * om * om * d_om5 : 0.f;
      const float d_a = -d_V * Vg / Va, d_b = -d_V * Vg / Vb;
      d_nl += d_a * (1.f - kk);
      const float d_nv = d_b * (1.f - kk);
      const float d_k = d_a * (1.f - nl) + d_b * (1.f - nv);
      float d_ar = 0.5f * d_k;
      float d_a2 = d_D / (kPiF * dd * dd);
      const float d_dd = (a2 * nh * nh + s2 > 1e-12f) ? -2.f * Dg / dd * d_D : 0.f;
      d_a2 += d_dd * nh * nh;
      const float d_nh = (ndh > 0.f && ndh < 1.f) ? d_dd * 2.f * a2 * nh : 0.f;
      const float d_s2 = d_dd;
      d_ar += 2.f * ar * d_a2;
      if (rough * rough > 1e-3f) d_q[7] += 2.f * rough * d_ar;
      float d_n[3], d_h[3], d_l[3], d_v[3], dc[3], t3[3];
      for (int k = 0; k < 3; ++k) dc[k] = 2.f * cxh[k] * d_s2;
      cross3f(h, dc, d_n);          // c = n x h: dL/dn = h x dc, dL/dh = dc x n
      cross3f(dc, n, d_h);
      for (int k = 0; k < 3; ++k) {
        d_n[k] += d_nh * h[k];
        d_h[k] += d_nh * n[k] + d_vh * v[k];
        d_v[k] = d_vh * h[k];
        d_l[k] = 0.f;
      }
      if (ndv > 1e-4f)
        for (int k = 0; k < 3; ++k) { d_n[k] += d_nv * v[k]; d_v[k] += d_nv * n[k]; }
      if (ndl > 0.f)
        for (int k = 0; k < 3; ++k) { d_n[k] += d_nl * l[k]; d_l[k] += d_nl * n[k]; }
      if (has_h) {
        normalize_bwd(h, ihl, d_h, t3);
        for (int k = 0; k < 3; ++k) { d_l[k] += t3[k]; d_v[k] += t3[k]; }
      } else {
        for (int k = 0; k < 3; ++k) d_n[k] += d_h[k];
      }
      normalize_bwd(n, 1.f / nn, d_n, t3);
      for (int k = 0; k < 3; ++k) d_q[1 + k] += t3[k];
      float d_lv[3], d_vv[3], d_xw[3], d_xc[3];
      normalize_bwd(l, il, d_l, d_lv);
      normalize_bwd(v, iv, d_v, d_vv);
      for (int k = 0; k < 3; ++k) d_xw[k] = -d_lv[k] - d_vv[k];
      for (int j = 0; j < 3; ++j) d_xc[j] = cam.R[3 * j] * d_xw[0] + cam.R[3 * j + 1] * d_xw[1] + cam.R[3 * j + 2] * d_xw[2];
      d_q[0] += d_xc[0] * ax + d_xc[1] * ay + d_xc[2];
    }
    // q_c = G_c / A
    for (int c = 0; c < 14; ++c) {
      dG[c] = d_q[c] * iA;
      dA -= d_q[c] * q[c] * iA;
    }
    dG[14] = dA;
  }
  // upstream gradient on the G-buffer itself (losses on the rasterised property images):
  // added to what reaches the G-buffer through rgb, on covered and uncovered pixels alike
  if (grad_gbuf_in != nullptr) {
    const float4* ip = reinterpret_cast<const float4*>(grad_gbuf_in + i * 16);
    for (int q = 0; q < 4; ++q) {
      const float4 v = ip[q];
      dG[4 * q] += v.x; dG[4 * q + 1] += v.y; dG[4 * q + 2] += v.z; dG[4 * q + 3] += v.w;
    }
  }
  float4* op = reinterpret_cast<float4*>(grad_gbuf + i * 16);
  for (int q = 0; q < 4; ++q) op[q] = make_float4(dG[4 * q], dG[4 * q + 1], dG[4 * q + 2], dG[4 * q + 3]);
}

// ---- a7 backward ----------------------------------------------------------------------------------------
// One CTA of 256 threads per tile, one thread per pixel (a warp = an 8x4 block, as in the one-slot forward walk).
// With Phi_i(p) = <dG(p), ch_i> (the upstream gradients dotted with entry i's channel vector, all lights, plus
// dG_A), the pixel's contribution to the loss is sum_i w_i Phi_i, w_i = T_i alpha_i, hence
//   dL / d alpha_i = T_i Phi_i - (sum_{j > i} w_j Phi_j) / (1 - alpha_i)        (one running suffix per pixel)
//   dL / d ch_i[c] = w_i dG[c].
// Phase A walks the list forward (same alpha rule and stop rule as the forward pass) to find where the pixel
// stopped and its final T; phase B walks back to front, dividing T by (1 - alpha_i) to recover T_i.
constexpr int kBwdBatch = 128;
struct BwdEntry {
  float4 ra, rb;      // (pix.x, pix.y, depth, -), (conic a, b, c unscaled, opacity)
};

template <int LB>
__global__ void __launch_bounds__(256)
composite_backward_kernel(CamParams cam, int n_lights, const uint2* __restrict__ ranges, const uint32_t* __restrict__ tile_order,
                          const uint32_t* __restrict__ sorted_vals, const float4* __restrict__ rec_a,
                          const float4* __restrict__ rec_b, const float4* __restrict__ attr,
                          const float4* __restrict__ mlp_out, int mlp_stride, const float* __restrict__ grad_gbuf,
                          int64_t npix, float* __restrict__ g_opacity, float* __restrict__ g_mean2d,
                          float* __restrict__ g_conic, float* __restrict__ g_depth, float* __restrict__ g_attr,
                          float* __restrict__ g_mlp_out, int64_t n) {
  __shared__ float4 s_a[kBwdBatch], s_b[kBwdBatch];
  __shared__ uint32_t s_g[kBwdBatch];
  __shared__ int s_last;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tile = (int)tile_order[blockIdx.x];   // longest lists first (the forward's work order): a short tail
  const int tx = tile % cam.tiles_x, ty = tile / cam.tiles_x;
  const int px = tx * kTile + (warp & 1) * 8 + (lane & 7), py = ty * kTile + (warp >> 1) * 4 + (lane >> 3);
  const bool inside = px < cam.width && py < cam.height;
  const int64_t pidx = (int64_t)min(py, cam.height - 1) * cam.width + min(px, cam.width - 1);
  // centre and half size of the warp's 8 x 4 pixel block: entries whose alpha >= 1/255 support box (rec_a.w, the
  // half-extents the forward walk culls with) misses the block are skipped by the whole warp, as in the forward
  const float bcx = (float)(tx * kTile + (warp & 1) * 8) + 3.5f, bcy = (float)(ty * kTile + (warp >> 1) * 4) + 1.5f;
  const uint2 range = ranges[tile];
  const int n_entries = (int)(range.y - range.x);
  constexpr float kInvLog2e = 0.6931471805599453f;   // rec_b holds the conic scaled by -log2(e)/2, -log2(e), -log2(e)/2
  // upstream gradients of this pixel: light-independent channels summed over the lights, MLP channels per light
  float dGs[11];   // depth, n3, b3, rough, metal, sss, A
  float dGl[LB][4];
  float dGT = 0.f;  // final transmittance (channel 15): non-zero only with an upstream gradient on the G-buffer
  for (int c = 0; c < 11; ++c) dGs[c] = 0.f;
  for (int l = 0; l < LB; ++l)
    for (int c = 0; c < 4; ++c) dGl[l][c] = 0.f;
  if (inside) {
    for (int l = 0; l < LB; ++l) {
      if (l >= n_lights) break;
      const float* gp = grad_gbuf + ((int64_t)l * npix + pidx) * 16;
      for (int c = 0; c < 10; ++c) dGs[c] += gp[c];
      dGs[10] += gp[14];
      dGT += gp[15];
      for (int c = 0; c < 4; ++c) dGl[l][c] = gp[10 + c];
    }
  }
  if (tid == 0) s_last = 0;
  __syncthreads();
  // ---- phase A: forward walk -> index after the last blended entry, T behind it ------------------
  float T = 1.f;
  int last = 0;
  bool done = !inside;
  for (int b0 = 0; b0 < n_entries; b0 += kBwdBatch) {
    if (__syncthreads_and(done)) break;
    const int cnt = min(kBwdBatch, n_entries - b0);
    if (tid < cnt) {
      const uint32_t gid = sorted_vals[range.x + b0 + tid];
      s_a[tid] = rec_a[gid];
      s_b[tid] = rec_b[gid];
    }
    __syncthreads();
    for (int c0 = 0; c0 < cnt; c0 += 32) {
      // cull 32 entries at a time (lane <-> entry), then walk the hits in list order
      bool hit = false;
      if (c0 + lane < cnt) {
        const float4 ra = s_a[c0 + lane];
        const float2 ext = __half22float2(*reinterpret_cast<const __half2*>(&ra.w));
        hit = fabsf(ra.x - bcx) <= ext.x + 3.5f && fabsf(ra.y - bcy) <= ext.y + 1.5f;
      }
      unsigned m = __ballot_sync(0xFFFFFFFFu, hit);
      while (m) {
        const int j = c0 + __ffs(m) - 1;
        m &= m - 1;
        const float4 ra = s_a[j], rb = s_b[j];
        const float dx = (float)px - ra.x, dy = (float)py - ra.y;
        const float p2 = fmaf(fmaf(rb.y, dy, rb.x * dx), dx, rb.z * dy * dy);   // log2(e) * power, as in the forward walk
        float al;
        asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(al) : "f"(p2));
        al = fminf(kAlphaMax, rb.w * al);
        if (!done && p2 <= 0.f && al >= kAlphaMin) {
          const float Tn = T * (1.f - al);
          if (Tn < kTMin) {
            done = true;
          } else {
            T = Tn;
            last = b0 + j + 1;
          }
        }
      }
    }
  }
  atomicMax(&s_last, last);
  __syncthreads();
  const int max_last = s_last;
  // destination of value k = 32 q + lane of an entry (see the reduction below): base pointer and per-Gaussian stride
  float* dst[(16 + 4 * LB + 31) / 32];
  int dst_stride[(16 + 4 * LB + 31) / 32];
#pragma unroll
  for (int q = 0; q < (16 + 4 * LB + 31) / 32; ++q) {
    const int k = 32 * q + lane;
    dst[q] = nullptr;
    dst_stride[q] = 0;
    if (k == 0) { dst[q] = g_opacity; dst_stride[q] = 1; }
    else if (k <= 2) { dst[q] = g_mean2d + (k - 1); dst_stride[q] = 2; }
    else if (k <= 5) { dst[q] = g_conic + (k - 3); dst_stride[q] = 3; }
    else if (k == 6) { dst[q] = g_depth; dst_stride[q] = 1; }
    else if (k <= 15) { dst[q] = g_attr + (k - 7); dst_stride[q] = 9; }
    else if (k < 16 + 4 * LB && (k - 16) / 4 < n_lights) {
      dst[q] = g_mlp_out + (size_t)((k - 16) / 4) * n * 4 + ((k - 16) & 3);
      dst_stride[q] = 4;
    }
  }
  // ---- phase B: back to front ---------------------------------------------------------------------
  // R = sum_{j > i} w_j Phi_j, started at dGT T_final: the final transmittance T_final = prod_j (1 - alpha_j) has
  // d T_final / d alpha_i = -T_final / (1 - alpha_i), the form of the suffix term below
  float R = dGT * T;
  for (int b1 = max_last; b1 > 0; b1 -= kBwdBatch) {
    const int b0 = max(0, b1 - kBwdBatch), cnt = b1 - b0;
    __syncthreads();
    if (tid < cnt) {
      const uint32_t gid = sorted_vals[range.x + b0 + tid];
      s_g[tid] = gid;
      s_a[tid] = rec_a[gid];
      s_b[tid] = rec_b[gid];
    }
    __syncthreads();
    for (int c0 = ((cnt - 1) >> 5) << 5; c0 >= 0; c0 -= 32) {
     bool hit = false;
     if (c0 + lane < cnt) {
       const float4 ra = s_a[c0 + lane];
       const float2 ext = __half22float2(*reinterpret_cast<const __half2*>(&ra.w));
       hit = fabsf(ra.x - bcx) <= ext.x + 3.5f && fabsf(ra.y - bcy) <= ext.y + 1.5f;
     }
     unsigned hits = __ballot_sync(0xFFFFFFFFu, hit);
     while (hits) {   // the hits of the chunk, last entry first
      const int hb = 31 - __clz(hits);
      hits &= ~(1u << hb);
      const int j = c0 + hb;
      const float4 ra = s_a[j];
      const float4 rb = s_b[j];
      const uint32_t gid = s_g[j];
      const float dx = (float)px - ra.x, dy = (float)py - ra.y;
      const float p2 = fmaf(fmaf(rb.y, dy, rb.x * dx), dx, rb.z * dy * dy);
      float e;
      asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(p2));
      const float araw = rb.w * e;
      const float al = fminf(kAlphaMax, araw);
      const bool blended = inside && (b0 + j) < last && p2 <= 0.f && al >= kAlphaMin;
      float w = 0.f, d_alpha = 0.f;
      if (!__any_sync(0xFFFFFFFFu, blended)) continue;
      // channel vector of the entry: warp-uniform loads (L1 / L2 hits)
      const float4 a0 = attr[3 * (size_t)gid], a1 = attr[3 * (size_t)gid + 1], a2 = attr[3 * (size_t)gid + 2];
      float4 mo[LB];
      for (int l = 0; l < LB; ++l) mo[l] = l < n_lights ? mlp_out[(size_t)gid * mlp_stride + l] : make_float4(0.f, 0.f, 0.f, 0.f);
      if (blended) {
        const float Ti = T / (1.f - al);       // transmittance in front of the entry
        w = Ti * al;
        float phi = dGs[0] * ra.z + dGs[1] * a0.x + dGs[2] * a0.y + dGs[3] * a0.z + dGs[4] * a1.x + dGs[5] * a1.y +
                    dGs[6] * a1.z + dGs[7] * a0.w + dGs[8] * a1.w + dGs[9] * a2.x + dGs[10];
        for (int l = 0; l < LB; ++l) phi += dGl[l][0] * mo[l].x + dGl[l][1] * mo[l].y + dGl[l][2] * mo[l].z + dGl[l][3] * mo[l].w;
        d_alpha = Ti * phi - R / (1.f - al);
        R += w * phi;
        T = Ti;
      }
      // ---- sums over the pixels of the warp, then one atomic per value -----------------------------
      {
        // alpha = o e^power (unclamped); power = -(a dx^2 + c dy^2) / 2 - b dx dy
        const bool unclamped = araw < kAlphaMax;
        const float d_o = (blended && unclamped) ? d_alpha * e : 0.f;
        const float d_pow = (blended && unclamped) ? d_alpha * al : 0.f;
        const float ca = -2.f * kInvLog2e * rb.x, cb = -kInvLog2e * rb.y, cc = -2.f * kInvLog2e * rb.z;
        // value k of the entry: 0 opacity, 1-2 mean, 3-5 conic, 6 depth, 7-15 attributes, 16 + 4 l + c MLP output c of
        // light l.  Groups of 32 values are summed over the 32 pixels of the warp with a halving exchange (31
        // shuffles per group instead of 5 per value); lane k of group q ends up with the sum of value 32 q + k and
        // adds it to its own destination: the atomics of an entry are issued by 16 + 4 LB lanes at once.
        constexpr int NG = (16 + 4 * LB + 31) / 32;
        float vals[32 * NG];
        vals[0] = d_o;
        vals[1] = d_pow * (ca * dx + cb * dy);      // d power / d pix_x
        vals[2] = d_pow * (cc * dy + cb * dx);
        vals[3] = d_pow * (-0.5f * dx * dx);         // d power / d conic a, b, c
        vals[4] = d_pow * (-dx * dy);
        vals[5] = d_pow * (-0.5f * dy * dy);
#pragma unroll
        for (int c = 0; c < 10; ++c) vals[6 + c] = w * dGs[c];
#pragma unroll
        for (int l = 0; l < LB; ++l)
#pragma unroll
          for (int c = 0; c < 4; ++c) vals[16 + 4 * l + c] = w * dGl[l][c];
#pragma unroll
        for (int k = 16 + 4 * LB; k < 32 * NG; ++k) vals[k] = 0.f;
#pragma unroll
        for (int q = 0; q < NG; ++q) {
#pragma unroll
          for (int half = 16; half >= 1; half >>= 1) {
            const bool up = (lane & half) != 0;
#pragma unroll
            for (int i = 0; i < half; ++i) {
              const float send = up ? vals[32 * q + i] : vals[32 * q + i + half];
              const float recv = __shfl_xor_sync(0xFFFFFFFFu, send, half);
              vals[32 * q + i] = (up ? vals[32 * q + i + half] : vals[32 * q + i]) + recv;
            }
          }
          if (dst[q] != nullptr) atomicAdd(dst[q] + (size_t)gid * dst_stride[q], vals[32 * q]);
        }
      }
     }
    }
  }
}

// ---- a2 backward: input rows, and the fp32 CUDA-core path ------------------------------------------
// The MLP input row of (Gaussian, light), as the forward kernel assembles it.
// x[0 .. 39]: the 40 inputs of the paper; every index is a compile-time constant once the loops are unrolled, so a
// caller's `float x[40]` stays in registers
__device__ __forceinline__ void mlp_input_geo(const sssgs_gaussians& g, int64_t i, const float* cam_pos,
                                              const float* light_pos, float* x) {
  const float mu[3] = {g.means[3 * i], g.means[3 * i + 1], g.means[3 * i + 2]};
#pragma unroll
  for (int k = 0; k < 3; ++k) x[k] = g.normals[3 * i + k];
  const float sgn = g.rotations[4 * i] < 0.f ? -1.f : 1.f;
  x[3] = sgn * g.rotations[4 * i];
  x[4] = sgn * g.rotations[4 * i + 1];
#pragma unroll
  for (int k = 0; k < 3; ++k) x[5 + k] = g.scales[3 * i + k];
  float wi[3], wo[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) { wi[k] = light_pos[k] - mu[k]; wo[k] = cam_pos[k] - mu[k]; }
  const float d = sqrtf(dot3f(wi, wi)), dn = sqrtf(dot3f(wo, wo));
#pragma unroll
  for (int k = 0; k < 3; ++k) { x[8 + k] = wi[k] / d; x[11 + k] = wo[k] / dn; }
  x[14] = d;
  const int nc = (g.vis_sh_degree + 1) * (g.vis_sh_degree + 1);
  float v = 0.2820948f * g.vis_sh[nc * i];
  if (g.vis_sh_degree >= 1)
    v += 0.4886025f * (g.vis_sh[nc * i + 1] * x[9] + g.vis_sh[nc * i + 2] * x[10] + g.vis_sh[nc * i + 3] * x[8]);
  x[15] = fminf(1.f, fmaxf(0.f, v));
#pragma unroll
  for (int k = 0; k < 4; ++k)
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      float s, c;
      sincospif((float)(1 << k) * mu[a], &s, &c);
      x[16 + 6 * k + a] = s;
      x[16 + 6 * k + 3 + a] = c;
    }
}
__device__ __forceinline__ void mlp_input_row(const sssgs_gaussians& g, int64_t i, const float* cam_pos,
                                              const float* light_pos, float* x) {
  mlp_input_geo(g, i, cam_pos, light_pos, x);
  for (int k = 0; k < g.feat_dim; ++k) x[40 + k] = g.feat[(int64_t)g.feat_dim * i + k];
}

// ---- a1 backward: dL/d(input row) -> the Gaussian -----------------------------------------------------------
// Where the gradients that arrive at the MLP's inputs go (all outputs are accumulated with atomics; NULL feat /
// vis_sh = the whole step is off).
struct InputGrads {
  float* means;      // [n][3]
  float* scales;     // [n][3]
  float* rotations;  // [n][4]
  float* attr;       // [n][9]: the normal is entries 0..2
  float* feat;       // [n][F]
  float* vis_sh;     // [n][ncoef]
};
// The row's quantities the Jacobian of mlp_input_geo needs, recomputed from the Gaussian (L2-hot).
struct InputCtx {
  float mu[3], wi[3], wo[3], di, dn, sgn, sh[4];
  bool v_free, deg1;
};
__device__ __forceinline__ void input_ctx(const sssgs_gaussians& g, int64_t i, const float* cam_pos, const float* light_pos,
                                          InputCtx& c) {
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    c.mu[k] = g.means[3 * i + k];
    c.wi[k] = light_pos[k] - c.mu[k];
    c.wo[k] = cam_pos[k] - c.mu[k];
  }
  c.di = sqrtf(dot3f(c.wi, c.wi));
  c.dn = sqrtf(dot3f(c.wo, c.wo));
#pragma unroll
  for (int k = 0; k < 3; ++k) { c.wi[k] /= c.di; c.wo[k] /= c.dn; }
  c.sgn = g.rotations[4 * i] < 0.f ? -1.f : 1.f;
  c.deg1 = g.vis_sh_degree >= 1;
  const int nc = c.deg1 ? 4 : 1;
  c.sh[0] = g.vis_sh[nc * i];
#pragma unroll
  for (int k = 1; k < 4; ++k) c.sh[k] = c.deg1 ? g.vis_sh[nc * i + k] : 0.f;
  const float v = 0.2820948f * c.sh[0] + 0.4886025f * (c.sh[1] * c.wi[1] + c.sh[2] * c.wi[2] + c.sh[3] * c.wi[0]);
  c.v_free = v > 0.f && v < 1.f;
}
// Partial sums of one thread's columns of a row.
struct InputAcc { float mu[3], nrm[3], q[2], s[3], sh[4]; };
__device__ __forceinline__ void input_acc_zero(InputAcc& a) {
#pragma unroll
  for (int k = 0; k < 3; ++k) a.mu[k] = a.nrm[k] = a.s[k] = 0.f;
  a.q[0] = a.q[1] = 0.f;
#pragma unroll
  for (int k = 0; k < 4; ++k) a.sh[k] = 0.f;
}
// d(mu) of a gradient dw arriving at the unit vector w = (p - mu) / dist
__device__ __forceinline__ void unit_dir_back(const float* w, float dist, const float* dw, float* dmu) {
  const float proj = dot3f(w, dw);
#pragma unroll
  for (int k = 0; k < 3; ++k) dmu[k] -= (dw[k] - w[k] * proj) / dist;
}
// Columns c0 .. c0 + cnt - 1 (< 40) of dL/d(input row): v[k] is the gradient of column c0 + k.
__device__ __forceinline__ void input_cols_back(const InputCtx& c, int c0, int cnt, const float* v, InputAcc& a) {
  float dwi[3] = {0.f, 0.f, 0.f}, dwo[3] = {0.f, 0.f, 0.f};
  bool any_wi = false, any_wo = false;
  for (int k = 0; k < cnt; ++k) {
    const int col = c0 + k;
    const float x = v[k];
    if (col < 3) a.nrm[col] += x;
    else if (col < 5) a.q[col - 3] += c.sgn * x;
    else if (col < 8) a.s[col - 5] += x;
    else if (col < 11) { dwi[col - 8] += x; any_wi = true; }
    else if (col < 14) { dwo[col - 11] += x; any_wo = true; }
    else if (col == 14) {
#pragma unroll
      for (int q = 0; q < 3; ++q) a.mu[q] -= x * c.wi[q];          // d = |L - mu|
    } else if (col == 15) {
      if (c.v_free) {                                               // the clamp to [0, 1] is a constant elsewhere
        a.sh[0] += 0.2820948f * x;
        if (c.deg1) {
          a.sh[1] += 0.4886025f * c.wi[1] * x;
          a.sh[2] += 0.4886025f * c.wi[2] * x;
          a.sh[3] += 0.4886025f * c.wi[0] * x;
          dwi[0] += 0.4886025f * c.sh[3] * x;
          dwi[1] += 0.4886025f * c.sh[1] * x;
          dwi[2] += 0.4886025f * c.sh[2] * x;
          any_wi = true;
        }
      }
    } else if (col < 40) {                                          // Fourier encoding of mu
      const int j = col - 16, oct = j / 6, w6 = j - 6 * oct, ax = w6 % 3;
      const float fr = (float)(1 << oct);
      float sn, cs;
      sincospif(fr * c.mu[ax], &sn, &cs);
      a.mu[ax] += (w6 < 3 ? cs : -sn) * fr * kPiF * x;
    }
  }
  if (any_wi) unit_dir_back(c.wi, c.di, dwi, a.mu);
  if (any_wo) unit_dir_back(c.wo, c.dn, dwo, a.mu);
}
__device__ __forceinline__ void input_acc_flush(const InputAcc& a, const InputGrads& o, int64_t i, bool deg1) {
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    if (a.mu[k] != 0.f) atomicAdd(&o.means[3 * i + k], a.mu[k]);
    if (a.nrm[k] != 0.f) atomicAdd(&o.attr[9 * i + k], a.nrm[k]);
    if (a.s[k] != 0.f) atomicAdd(&o.scales[3 * i + k], a.s[k]);
  }
  if (a.q[0] != 0.f) atomicAdd(&o.rotations[4 * i], a.q[0]);
  if (a.q[1] != 0.f) atomicAdd(&o.rotations[4 * i + 1], a.q[1]);
  const int nc = deg1 ? 4 : 1;
#pragma unroll
  for (int k = 0; k < 4; ++k)
    if (k < nc && a.sh[k] != 0.f) atomicAdd(&o.vis_sh[nc * i + k], a.sh[k]);
}
// One call per (row, run of columns): geometric columns through the Jacobian, feature columns straight through.
__device__ __forceinline__ void input_row_back(const sssgs_gaussians& g, int64_t i, const float* cam_pos, const float* light_pos,
                                               int c0, int cnt, const float* v, const InputGrads& o) {
  bool any = false;
  for (int k = 0; k < cnt; ++k) any = any || v[k] != 0.f;
  if (!any) return;
  const int geo = c0 < 40 ? min(cnt, 40 - c0) : 0;
  if (geo > 0) {
    InputCtx ctx;
    input_ctx(g, i, cam_pos, light_pos, ctx);
    InputAcc acc;
    input_acc_zero(acc);
    input_cols_back(ctx, c0, geo, v, acc);
    input_acc_flush(acc, o, i, ctx.deg1);
  }
  for (int k = geo; k < cnt; ++k) {
    const int f = c0 + k - 40;
    if (f < g.feat_dim && v[k] != 0.f) atomicAdd(&o.feat[(int64_t)g.feat_dim * i + f], v[k]);
  }
}

// Layer table of the MLP in the caller's parameter packing (sssgs_mlp.params, fp32).
struct BwdLayer { int w, b, out, in, src, kind; };   // src: index of the layer whose output feeds this one (-1: x)
struct BwdNet {
  int n_layers, in_dim, activation, trunk_last;
  float slope;
  BwdLayer L[SSSGS_MAX_TRUNK + SSSGS_MAX_INC_HIDDEN + 2];
};
enum { K_HIDDEN = 0, K_SSS = 1, K_INC_OUT = 2 };

constexpr int kBR = 16;    // rows of a tile
constexpr int kWS = 132;   // row stride of the staged weight matrix (floats): 16-byte aligned rows, conflict-free LDS.128 down a column

// Rows of the batch whose dL/d(mlp_out) is not all zero (a Gaussian no pixel blended gets no gradient: 88 % of the
// rows of a large scene), compacted into a list; order is arbitrary (the sums below are atomics anyway).
__global__ void __launch_bounds__(256)
bwd_rows_kernel(const float4* __restrict__ g_mlp_out, int64_t total, uint32_t* __restrict__ list, uint32_t* __restrict__ count) {
  // count[0] = rows listed, count[1] = bits of the largest |dL/d(mlp_out)| (non-negative floats order as integers)
  for (int64_t base = (int64_t)blockIdx.x * 256; base < total; base += (int64_t)gridDim.x * 256) {
    const int64_t idx = base + threadIdx.x;
    bool on = false;
    uint32_t mx = 0u;
    if (idx < total) {
      const float4 v = g_mlp_out[idx];
      on = v.x != 0.f || v.y != 0.f || v.z != 0.f || v.w != 0.f;
      mx = __float_as_uint(fmaxf(fmaxf(fabsf(v.x), fabsf(v.y)), fmaxf(fabsf(v.z), fabsf(v.w))));
      if (mx >= 0x7F800000u) mx = 0u;   // inf / NaN do not set the scale
    }
    mx = __reduce_max_sync(0xffffffffu, mx);
    if ((threadIdx.x & 31) == 0 && mx > 0u) atomicMax(count + 1, mx);
    const unsigned m = __ballot_sync(0xffffffffu, on);
    const int lane = threadIdx.x & 31;
    unsigned at = 0;
    if (lane == 0 && m) at = atomicAdd(count, (unsigned)__popc(m));
    at = __shfl_sync(0xffffffffu, at, 0);
    if (on) list[at + __popc(m & ((1u << lane) - 1u))] = (uint32_t)idx;
  }
}

__device__ __forceinline__ float dot4(const float4 a, const float4 b, float s) {
  return fmaf(a.w, b.w, fmaf(a.z, b.z, fmaf(a.y, b.y, fmaf(a.x, b.x, s))));
}

// MLP backward (step a2 differentiated), fp32 on the CUDA cores.  blockIdx.y = the layer whose weight gradient this
// CTA accumulates (64 register accumulators per thread cover its out x in <= 128 x 128 matrix); blockIdx.x strides
// over tiles of kBR listed rows.  Per tile: inputs (recomputed from the Gaussian, as the forward kernel does), the
// forward pass through every layer (activations stay in shared memory), the delta recursion from the two heads down
// to the target layer, and  dW += delta^T h,  db += sum delta.  Each layer's weights are staged in shared memory
// once per tile and pass.  The accumulators go to global memory once, with atomics, when the CTA has no tiles left.
__global__ void __launch_bounds__(256, 1)
mlp_backward_kernel(sssgs_gaussians g, BwdNet net, const float* __restrict__ params, CamParams cam, LightBatch lights,
                    int64_t n, const uint32_t* __restrict__ list, const uint32_t* __restrict__ count,
                    const float* __restrict__ g_mlp_out, float* __restrict__ g_params, InputGrads ig) {
  extern __shared__ __align__(16) float bw_smem[];
  float* sW = bw_smem;                           // [128][kWS]
  float* sGA = sW + 128 * kWS;                   // [kBR][128] gradient wrt a trunk layer's output
  float* sGB = sGA + kBR * 128;                  // [kBR][128] ... an incident-head layer's output
  float* sD = sGB + kBR * 128;                   // [kBR][128] delta of the current layer
  float* sGo = sD + kBR * 128;                   // [kBR][4]   dL/d(mlp_out) of the rows
  float* sAct = sGo + kBR * 4;                   // [n_layers + 1][kBR][128]: x, then each layer's output
  const int tid = threadIdx.x;
  const int target = blockIdx.y;
  const BwdLayer T = net.L[target];
  const int trunk_last = net.trunk_last;
  const unsigned nrows = *count;
  const unsigned ntiles = (nrows + kBR - 1) / kBR;
  float acc[8][8];
  float accb[8];
#pragma unroll
  for (int a = 0; a < 8; ++a) {
    accb[a] = 0.f;
#pragma unroll
    for (int b = 0; b < 8; ++b) acc[a][b] = 0.f;
  }
  const int rg = tid >> 6, oc = tid & 63;        // forward / delta recursion: rows 4 rg .. 4 rg + 3
  const int to = tid >> 4, ti = tid & 15;        // dW: outputs 4 to + {0..3}, 64 + 4 to + {0..3}; inputs likewise with ti
  bool any = false;

  auto stage_weights = [&](const BwdLayer& L) {   // sW[o][k] = W[o][k], zero outside out x in
    __syncthreads();
    for (int idx = tid; idx < 128 * 128; idx += 256) {
      const int o = idx >> 7, k = idx & 127;
      sW[o * kWS + k] = (o < L.out && k < L.in) ? params[L.w + (size_t)o * L.in + k] : 0.f;
    }
    __syncthreads();
  };

  for (unsigned tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    any = true;
    __syncthreads();
    // ---- rows of the tile: inputs and upstream gradients ----
    for (int idx = tid; idx < kBR * 128; idx += 256) sAct[idx] = 0.f;
    __syncthreads();
    if (tid < kBR) {
      const unsigned r = tile * kBR + tid;
      float4 go = make_float4(0.f, 0.f, 0.f, 0.f);
      if (r < nrows) {
        const uint32_t idx = list[r];
        const int64_t i = idx % n;
        const int l_idx = (int)(idx / n);
        go = reinterpret_cast<const float4*>(g_mlp_out)[idx];
        mlp_input_row(g, i, cam.pos, lights.l[l_idx].pos, sAct + tid * 128);
      }
      reinterpret_cast<float4*>(sGo)[tid] = go;
    }
    // ---- forward ----
    for (int l = 0; l < net.n_layers; ++l) {
      const BwdLayer L = net.L[l];
      stage_weights(L);
      const float* hin = sAct + (size_t)(L.src + 1) * kBR * 128;
      float* hout = sAct + (size_t)(l + 1) * kBR * 128;
      if (oc < L.out || L.out > 64) {
        float sum[4][2];
        const float b0 = oc < L.out ? params[L.b + oc] : 0.f, b1 = oc + 64 < L.out ? params[L.b + oc + 64] : 0.f;
#pragma unroll
        for (int r = 0; r < 4; ++r) sum[r][0] = b0, sum[r][1] = b1;
        const int in4 = (L.in + 3) & ~3;
        for (int k = 0; k < in4; k += 4) {
          const float4 w0 = *reinterpret_cast<const float4*>(sW + oc * kWS + k);
          const float4 w1 = *reinterpret_cast<const float4*>(sW + (oc + 64) * kWS + k);
#pragma unroll
          for (int r = 0; r < 4; ++r) {
            const float4 h = *reinterpret_cast<const float4*>(hin + (4 * rg + r) * 128 + k);
            sum[r][0] = dot4(h, w0, sum[r][0]);
            sum[r][1] = dot4(h, w1, sum[r][1]);
          }
        }
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
          for (int j = 0; j < 2; ++j) {
            const int o = oc + 64 * j;
            const float v = sum[r][j];
            float y;
            if (L.kind == K_HIDDEN) y = v > 0.f ? v : (net.activation == SSSGS_ACT_LEAKY_RELU ? net.slope * v : 0.f);
            else if (L.kind == K_SSS) y = 1.f / (1.f + expf(-v));
            else y = fmaxf(0.f, v);
            hout[(4 * rg + r) * 128 + o] = o < L.out ? y : 0.f;
          }
      } else {
#pragma unroll
        for (int r = 0; r < 4; ++r) hout[(4 * rg + r) * 128 + oc] = 0.f, hout[(4 * rg + r) * 128 + oc + 64] = 0.f;
      }
    }
    __syncthreads();
    for (int idx = tid; idx < kBR * 128; idx += 256) sGA[idx] = 0.f;
    // ---- delta recursion, from the last layer down to the target ----
    for (int l = net.n_layers - 1; l >= target; --l) {
      const BwdLayer L = net.L[l];
      const float* y = sAct + (size_t)(l + 1) * kBR * 128;
      const float* gout = l <= trunk_last ? sGA : sGB;
      __syncthreads();
      for (int idx = tid; idx < kBR * 128; idx += 256) {
        const int r = idx >> 7, o = idx & 127;
        float d = 0.f;
        if (o < L.out) {
          const float yy = y[idx];
          if (L.kind == K_SSS) d = sGo[4 * r + o] * yy * (1.f - yy);
          else if (L.kind == K_INC_OUT) d = yy > 0.f ? sGo[4 * r + 3] : 0.f;
          else d = gout[idx] * (yy > 0.f ? 1.f : (net.activation == SSSGS_ACT_LEAKY_RELU ? net.slope : 0.f));
        }
        sD[idx] = d;
      }
      if (l == target) break;
      if (L.src < 0) continue;
      stage_weights(L);     // (syncs: sD is complete)
      // gradient wrt the source layer's output: G[r][i] (+)= sum_o D[r][o] W[o][i]; thread: 4 rows x inputs 2 oc, 2 oc + 1
      float* gdst = L.src <= trunk_last ? sGA : sGB;
      const bool accumulate = L.src == trunk_last;      // both heads feed the last trunk layer
      float s2[4][2];
#pragma unroll
      for (int r = 0; r < 4; ++r) s2[r][0] = s2[r][1] = 0.f;
      const int out4 = (L.out + 3) & ~3;
      for (int o = 0; o < out4; o += 4) {
        float4 d4[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) d4[r] = *reinterpret_cast<const float4*>(sD + (4 * rg + r) * 128 + o);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float2 w = *reinterpret_cast<const float2*>(sW + (o + j) * kWS + 2 * oc);
#pragma unroll
          for (int r = 0; r < 4; ++r) {
            const float d = j == 0 ? d4[r].x : j == 1 ? d4[r].y : j == 2 ? d4[r].z : d4[r].w;
            s2[r][0] = fmaf(d, w.x, s2[r][0]);
            s2[r][1] = fmaf(d, w.y, s2[r][1]);
          }
        }
      }
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        float2* dst = reinterpret_cast<float2*>(gdst + (4 * rg + r) * 128 + 2 * oc);
        float2 v = make_float2(s2[r][0], s2[r][1]);
        if (accumulate) { const float2 old = *dst; v.x += old.x; v.y += old.y; }
        *dst = v;
      }
    }
    __syncthreads();
    // ---- a1: dL/dx = delta_0 W_0, pushed through the input assembly (CTAs of target 0 only) ----
    if (target == 0 && ig.feat != nullptr) {
      const BwdLayer L0 = net.L[0];
      stage_weights(L0);
      float s2[4][2];
#pragma unroll
      for (int r = 0; r < 4; ++r) s2[r][0] = s2[r][1] = 0.f;
      const int out4 = (L0.out + 3) & ~3;
      for (int o = 0; o < out4; o += 4) {
        float4 d4[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) d4[r] = *reinterpret_cast<const float4*>(sD + (4 * rg + r) * 128 + o);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float2 w = *reinterpret_cast<const float2*>(sW + (o + j) * kWS + 2 * oc);
#pragma unroll
          for (int r = 0; r < 4; ++r) {
            const float d = j == 0 ? d4[r].x : j == 1 ? d4[r].y : j == 2 ? d4[r].z : d4[r].w;
            s2[r][0] = fmaf(d, w.x, s2[r][0]);
            s2[r][1] = fmaf(d, w.y, s2[r][1]);
          }
        }
      }
#pragma unroll
      for (int r = 0; r < 4; ++r) *reinterpret_cast<float2*>(sGB + (4 * rg + r) * 128 + 2 * oc) = make_float2(s2[r][0], s2[r][1]);
      __syncthreads();
      // thread = (row, run of 8 columns)
      const int r = tid >> 4, c0 = (tid & 15) * 8;
      const unsigned ridx = tile * kBR + r;
      if (ridx < nrows && c0 < net.in_dim) {
        const uint32_t idx = list[ridx];
        float v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = c0 + k < net.in_dim ? sGB[r * 128 + c0 + k] : 0.f;
        input_row_back(g, (int64_t)(idx % n), cam.pos, lights.l[idx / n].pos, c0, min(8, net.in_dim - c0), v, ig);
      }
      __syncthreads();
    }
    // ---- dW[o][i] += sum_r D[r][o] h[r][i],  db[o] += sum_r D[r][o] ----
    const float* hsrc = sAct + (size_t)(T.src + 1) * kBR * 128;
#pragma unroll 2
    for (int r = 0; r < kBR; ++r) {
      const float4 d0 = *reinterpret_cast<const float4*>(sD + r * 128 + 4 * to);
      const float4 d1 = *reinterpret_cast<const float4*>(sD + r * 128 + 64 + 4 * to);
      const float4 h0 = *reinterpret_cast<const float4*>(hsrc + r * 128 + 4 * ti);
      const float4 h1 = *reinterpret_cast<const float4*>(hsrc + r * 128 + 64 + 4 * ti);
      const float dd[8] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
      const float hh[8] = {h0.x, h0.y, h0.z, h0.w, h1.x, h1.y, h1.z, h1.w};
#pragma unroll
      for (int a = 0; a < 8; ++a) {
        accb[a] += dd[a];
#pragma unroll
        for (int b = 0; b < 8; ++b) acc[a][b] = fmaf(dd[a], hh[b], acc[a][b]);
      }
    }
  }
  if (!any) return;
#pragma unroll
  for (int a = 0; a < 8; ++a) {
    const int o = (a < 4 ? 0 : 60) + 4 * to + a;      // a >= 4: 64 + 4 to + (a - 4)
    if (o >= T.out) continue;
    if (ti == 0) atomicAdd(&g_params[T.b + o], accb[a]);
#pragma unroll
    for (int b = 0; b < 8; ++b) {
      const int i = (b < 4 ? 0 : 60) + 4 * ti + b;
      if (i < T.in && acc[a][b] != 0.f) atomicAdd(&g_params[T.w + (size_t)o * T.in + i], acc[a][b]);
    }
  }
}

// ---- a2 backward on the tensor cores (tcgen05) -------------------------------------------------------
// For MLPs without incident-head hidden layers (every BASELINE config).  Per tile of 128 listed rows, a CTA
// recomputes the forward pass with the forward kernel's arithmetic (binary16 operands, fp32 accumulators in
// tensor memory, A operand from tensor memory), runs the delta recursion  G_{l-1} = delta_l W_l  as
// tcgen05.mma with the SAME shared-memory weight tile read MN-major (B[n][k] = W_l[k][n]: no transposed
// copy), and accumulates the weight gradient of ONE layer (blockIdx.y)  dW_t += delta_t^T h_{t-1}  over all
// of its tiles in 128 tensor-memory columns, both operands MN-major from shared memory (the 128 rows of the
// tile are the K dimension).  dL/d(mlp_out) is scaled by a power of two (largest magnitude of the batch in
// (0.5, 1]) so that the deltas fit binary16; the sums are un-scaled when they leave tensor memory.
namespace tc {

constexpr int kRowsT = 128;            // rows per tile = UMMA M (forward, recursion) = UMMA K (weight gradient)
constexpr int kTileBytes = 32768;      // one [128][128] 16-bit operand tile: two 64-column blocks of 16 KB
constexpr int kHeadTileBytes = 4096;   // head weights: [2 blocks][16 rows][128 B]
constexpr uint32_t kColDW = 0, kColD = 128, kColA = 256, kColAH = 320;   // tensor-memory columns

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {
  }
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t* w) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr),
               "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7]) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float* v) {
  uint32_t r[16];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    asm volatile("" : "+r"(r[i]));
    v[i] = __uint_as_float(r[i]);
  }
}
// asynchronous form: r[] is valid only after tmem_wait_ld(r)
__device__ __forceinline__ void tmem_ld16_async(uint32_t taddr, uint32_t* r) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_wait_ld(uint32_t* r) {
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 16; ++i) asm volatile("" : "+r"(r[i]));
}
// Walks this thread's (up to four) 16-column groups c0 = first + 32 i < n of an accumulator: f(r, c0, i) gets the 16
// columns as bits and the group index as a compile-time constant (state indexed by it stays in registers); the
// tensor-memory load of the next group is in flight while a group is processed.
template <typename Fn>
__device__ __forceinline__ void for_groups(uint32_t taddr, int first, int n, Fn f) {
  uint32_t r[2][16];
  if (first < n) tmem_ld16_async(taddr + first, r[0]);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int c0 = first + 32 * i;
    if (c0 >= n) break;
    tmem_wait_ld(r[i & 1]);
    if (i + 1 < 4 && c0 + 32 < n) tmem_ld16_async(taddr + c0 + 32, r[(i + 1) & 1]);
    f(r[i & 1], c0, i);
  }
}
__device__ __forceinline__ uint32_t pack_f16(float a, float b) {   // .lo = a, .hi = b, RNE, saturating
  uint32_t d;
  asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(b), "f"(a));
  return d;
}
__device__ __forceinline__ uint32_t elect_one() {
  uint32_t e;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(e));
  return e;
}
// Shared-memory operand descriptor, 128-byte swizzle, version 1.  K-major: rows of 128 B, 8-row groups `sbo`
// bytes apart (lbo unused).  MN-major: 64 MN elements contiguous (128 B) per K row, 8 K rows per 1024-byte atom,
// atoms `sbo` apart along K and `lbo` apart along MN.
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr >> 4) & 0x3FFFu);
  d |= (uint64_t)((lbo >> 4) & 0x3FFFu) << 16;
  d |= (uint64_t)((sbo >> 4) & 0x3FFFu) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}
// D = F32, A = B = F16, M = 128, N = n; a_mn / b_mn: operand is MN-major
__device__ __forceinline__ uint32_t make_idesc(int n, bool a_mn, bool b_mn) {
  return (1u << 4) | ((a_mn ? 1u : 0u) << 15) | ((b_mn ? 1u : 0u) << 16) | ((uint32_t)(n >> 3) << 17) |
         ((uint32_t)(kRowsT >> 4) << 24);
}
// The whole issuing warp runs these with warp-uniform operands; the instruction is predicated on one lane.
__device__ __forceinline__ void umma_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t desc_b, uint32_t idesc, uint32_t acc,
                                        uint32_t issue) {
  asm volatile(
      "{\n\t.reg .pred p, q;\n\t"
      "setp.ne.u32 p, %4, 0;\n\t"
      "setp.ne.u32 q, %5, 0;\n\t"
      "@q tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(tmem_d), "r"(tmem_a), "l"(desc_b), "r"(idesc), "r"(acc), "r"(issue) : "memory");
}
__device__ __forceinline__ void umma_ss(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t acc,
                                        uint32_t issue) {
  asm volatile(
      "{\n\t.reg .pred p, q;\n\t"
      "setp.ne.u32 p, %4, 0;\n\t"
      "setp.ne.u32 q, %5, 0;\n\t"
      "@q tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(acc), "r"(issue) : "memory");
}
__device__ __forceinline__ void umma_commit_if(uint32_t bar, uint32_t issue) {
  asm volatile(
      "{\n\t.reg .pred q;\n\t"
      "setp.ne.u32 q, %1, 0;\n\t"
      "@q tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}"
      ::"r"(bar), "r"(issue) : "memory");
}
// byte offset of element (row r, column c) of a [rows][128] 16-bit tile stored as two 64-column blocks
// `block_bytes` apart, rows of 128 B, 128-byte swizzle (16-byte chunk index xor row % 8)
__device__ __forceinline__ uint32_t tile_off(int r, int c, int block_bytes) {
  return (uint32_t)((c >> 6) * block_bytes + r * 128 + ((((c & 63) >> 3) ^ (r & 7)) << 4) + (c & 7) * 2);
}

// Layer table of the tensor-core backward: layers 0 .. n_trunk - 1 = trunk, layer n_trunk = the two heads as one
// 4-row layer (rows 0-2 SSS, row 3 incident light).
struct TcNet {
  int n_trunk, in_dim, k0_pad, activation;
  float slope;
  int out[SSSGS_MAX_TRUNK], in[SSSGS_MAX_TRUNK], w[SSSGS_MAX_TRUNK], b[SSSGS_MAX_TRUNK];   // caller's packing (floats)
  int sss_w, sss_b, inc_w, inc_b, head_in;
};

// blob: trunk tiles (32 KB each, K-major = [out row][in column]), head tile (4 KB), then biases fp32 [n_trunk + 1][128]
__global__ void __launch_bounds__(256)
bwd_pack_kernel(TcNet net, const float* __restrict__ params, uint8_t* __restrict__ blob) {
  const int L = net.n_trunk;
  const int total = L * 128 * 128 + 16 * 128 + (L + 1) * 128;
  for (int idx = blockIdx.x * 256 + threadIdx.x; idx < total; idx += gridDim.x * 256) {
    if (idx < L * 128 * 128) {
      const int l = idx >> 14, n = (idx >> 7) & 127, k = idx & 127;
      const float v = (n < net.out[l] && k < net.in[l]) ? params[net.w[l] + n * net.in[l] + k] : 0.f;
      *reinterpret_cast<__half*>(blob + (size_t)l * kTileBytes + tile_off(n, k, 16384)) = __float2half_rn(v);
    } else if (idx < L * 128 * 128 + 16 * 128) {
      const int j = idx - L * 128 * 128, n = j >> 7, k = j & 127;
      float v = 0.f;
      if (k < net.head_in) {
        if (n < 3) v = params[net.sss_w + n * net.head_in + k];
        else if (n == 3) v = params[net.inc_w + k];
      }
      *reinterpret_cast<__half*>(blob + (size_t)L * kTileBytes + tile_off(n, k, 2048)) = __float2half_rn(v);
    } else {
      const int j = idx - L * 128 * 128 - 16 * 128, l = j >> 7, n = j & 127;
      float v = 0.f;
      if (l < L) { if (n < net.out[l]) v = params[net.b[l] + n]; }
      else if (n < 3) v = params[net.sss_b + n];
      else if (n == 3) v = params[net.inc_b];
      reinterpret_cast<float*>(blob + (size_t)L * kTileBytes + kHeadTileBytes)[j] = v;
    }
  }
}

struct TcArgs {
  sssgs_gaussians g;
  TcNet net;
  CamParams cam;
  LightBatch lights;
  int64_t n;
  const uint32_t* list;        // rows of the batch with a gradient (index = light * n + Gaussian)
  const uint32_t* count;
  const uint32_t* gomax_bits;  // bits of max |dL/d(mlp_out)| over the batch
  const float* g_mlp_out;      // [n_lights][n][4]
  const uint8_t* blob;         // bwd_pack_kernel's output
  float* g_params;
  InputGrads ig;               // a1 backward (feat == nullptr: off)
};

__host__ __device__ inline int tc_smem_bytes(int n_trunk) {
  return n_trunk * kTileBytes + kHeadTileBytes + 2 * kTileBytes + (n_trunk + 1) * 128 * 4 + 64 + 1024;
}

// 256 threads: thread pair (row, half) = (tid % 128, tid / 128); the two halves of a row split every epilogue's
// 16-column groups alternately (warps w and w + 4 read the same 32 tensor-memory lanes).
__global__ void __launch_bounds__(256, 1) mlp_backward_tc_kernel(const __grid_constant__ TcArgs a) {
  extern __shared__ uint8_t tc_smem_raw[];
  uint8_t* sm = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(tc_smem_raw) + 1023) & ~(uintptr_t)1023);
  const TcNet& net = a.net;
  const int L = net.n_trunk;
  uint8_t* sW = sm;
  uint8_t* sDelta = sW + (size_t)L * kTileBytes + kHeadTileBytes;
  uint8_t* sH = sDelta + kTileBytes;
  float* sBias = reinterpret_cast<float*>(sH + kTileBytes);
  uint64_t* bars = reinterpret_cast<uint64_t*>(sBias + (L + 1) * 128);
  uint32_t* s_tmem = reinterpret_cast<uint32_t*>(bars + 2);
  const int tid = threadIdx.x, warp = tid >> 5;
  const int row = tid & 127, half = tid >> 7;   // this thread's row of the tile and its share of the column groups
  const int t = blockIdx.y;                      // target layer: t < L trunk, t == L the heads
  const uint32_t bar = smem_u32(bars);

  // ---- set-up: weights and biases into shared memory, operand tiles zeroed, tensor memory --------------
  {
    const uint4* src = reinterpret_cast<const uint4*>(a.blob);
    uint4* dst = reinterpret_cast<uint4*>(sW);
    const int nw = (L * kTileBytes + kHeadTileBytes) / 16;
    for (int i = tid; i < nw; i += 256) dst[i] = src[i];
    const float* bsrc = reinterpret_cast<const float*>(a.blob + (size_t)L * kTileBytes + kHeadTileBytes);
    for (int i = tid; i < (L + 1) * 128; i += 256) sBias[i] = bsrc[i];
    uint4* z = reinterpret_cast<uint4*>(sDelta);
    for (int i = tid; i < 2 * kTileBytes / 16; i += 256) z[i] = make_uint4(0u, 0u, 0u, 0u);
  }
  if (tid == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(s_tmem)), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  fence_proxy_async();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *s_tmem;
  const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
  const uint32_t tD = tmem + kColD, tA = tmem + kColA, tAH = tmem + kColAH, tDW = tmem + kColDW;
  const uint32_t sW_addr = smem_u32(sW), sDelta_addr = smem_u32(sDelta), sH_addr = smem_u32(sH);
  uint32_t phase = 0;

  const int k_t = t == 0 ? net.k0_pad : (t < L ? net.in[t] : net.head_in);   // K of the target layer (padded)
  const uint32_t nrows = *a.count;
  const uint32_t ntiles = (nrows + kRowsT - 1) / kRowsT;
  // power-of-two scale: the largest |dL/d(mlp_out)| of the batch lands in (0.5, 1]
  const uint32_t mbits = *a.gomax_bits;
  int e = (int)(mbits >> 23) - 127;
  e = e < -100 ? -100 : (e > 100 ? 100 : e);
  const float scale = __uint_as_float((uint32_t)(126 - e) << 23), inv_scale = __uint_as_float((uint32_t)(128 + e) << 23);
  const bool want_x = a.ig.feat != nullptr;
  const bool leaky = net.activation == SSSGS_ACT_LEAKY_RELU;
  const float neg_slope = leaky ? net.slope : 0.f;
  float db = 0.f;
  uint32_t tiles_done = 0;
#ifdef SSSGS_BWD_TIMELINE
  long long tl[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tl_t = clock64();
#define TL(i) do { const long long c_ = clock64(); tl[i] += c_ - tl_t; tl_t = c_; } while (0)
#else
#define TL(i) do {} while (0)
#endif

  // this thread's operand writes before the next MMAs: tensor memory always, shared memory (generic -> async proxy
  // fence) only when an operand tile was written since the last call
  auto publish = [&](bool smem_written) {
    tmem_wait_st();
    if (smem_written) fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
  };
  auto wait_mma = [&]() {
    TL(6);
    mbar_wait(bar, phase);
    phase ^= 1u;
    tc_fence_after();
    TL(7);
  };
  // 16 consecutive 16-bit values of this thread's row (columns c0 .. c0 + 15) into a shared-memory operand tile
  auto store_row16 = [&](uint8_t* tile, int c0, const uint32_t* w) {
    *reinterpret_cast<uint4*>(tile + tile_off(row, c0, 16384)) = make_uint4(w[0], w[1], w[2], w[3]);
    *reinterpret_cast<uint4*>(tile + tile_off(row, c0 + 8, 16384)) = make_uint4(w[4], w[5], w[6], w[7]);
  };

  for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    // ---- the rows of the tile: inputs (as the forward kernel assembles them) and upstream gradients ------
    const uint32_t ridx = tile * kRowsT + row;
    float4 go = make_float4(0.f, 0.f, 0.f, 0.f);
    const int F = a.g.feat_dim;
    int64_t gi = -1;
    uint32_t li = 0;
    if (ridx < nrows) {
      const uint32_t idx = a.list[ridx];
      li = idx / (uint32_t)a.n;
      gi = (int64_t)(idx - li * (uint32_t)a.n);
      go = reinterpret_cast<const float4*>(a.g_mlp_out)[idx];
    }
    const float4* fp = gi >= 0 ? reinterpret_cast<const float4*>(a.g.feat + gi * F) : nullptr;   // the row's feature
    auto feat4 = [&](int q) {   // features 4 q .. 4 q + 3
      return (fp != nullptr && 4 * q < F) ? fp[q] : make_float4(0.f, 0.f, 0.f, 0.f);
    };
    // Columns 0-47 (the 40 computed inputs, in registers, and the first 8 features) by half 0, the remaining
    // feature columns by half 1 (16-byte loads, four in flight): no input is computed twice.
    if (half == 0) {
      const float4 f0 = feat4(0), f1 = feat4(1);
      float e[40];
#pragma unroll
      for (int k = 0; k < 40; ++k) e[k] = 0.f;
      if (gi >= 0) mlp_input_geo(a.g, gi, a.cam.pos, a.lights.l[li].pos, e);
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        uint32_t w[8];
        if (c < 2) {
#pragma unroll
          for (int i = 0; i < 8; ++i) w[i] = pack_f16(e[16 * c + 2 * i], e[16 * c + 2 * i + 1]);
        } else {
#pragma unroll
          for (int i = 0; i < 4; ++i) w[i] = pack_f16(e[32 + 2 * i], e[33 + 2 * i]);
          w[4] = pack_f16(f0.x, f0.y); w[5] = pack_f16(f0.z, f0.w);
          w[6] = pack_f16(f1.x, f1.y); w[7] = pack_f16(f1.z, f1.w);
        }
        tmem_st8(tA + lane_off + (uint32_t)(8 * c), w);
        if (t == 0) store_row16(sH, 16 * c, w);
      }
    } else {
      for (int c = 3; 16 * c < net.k0_pad; ++c) {
        float4 f[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) f[j] = feat4(4 * c - 10 + j);
        uint32_t w[8];
#pragma unroll
        for (int j = 0; j < 4; ++j) { w[2 * j] = pack_f16(f[j].x, f[j].y); w[2 * j + 1] = pack_f16(f[j].z, f[j].w); }
        tmem_st8(tA + lane_off + (uint32_t)(8 * c), w);
        if (t == 0) store_row16(sH, 16 * c, w);
      }
    }
    publish(t == 0);
    TL(0);

    // ---- forward, trunk ----------------------------------------------------------------------------------
    uint32_t mask[4][4];   // ReLU decisions: layer (<= 4 on this path), this thread's column group; registers
#pragma unroll
    for (int l = 0; l < 4; ++l) {
      if (l >= L) break;
      const int kl = l == 0 ? net.k0_pad : net.in[l], nl = net.out[l];
      if (warp == 0) {
        const uint32_t issue = elect_one();
        const uint32_t idesc = make_idesc(nl, false, false);
        for (int ks = 0; ks < kl / 16; ++ks)
          umma_ts(tD, tA + ks * 8, make_desc(sW_addr + l * kTileBytes + (ks >> 2) * 16384 + (ks & 3) * 32, 16, 1024), idesc,
                  ks > 0, issue);
        umma_commit_if(bar, issue);
      }
      wait_mma();
#pragma unroll
      for (int q = 0; q < 4; ++q) mask[l][q] = 0u;
      for_groups(tD + lane_off, 16 * half, nl, [&](const uint32_t* r, int c0, int gi_) {
        float v[16];
        uint32_t bits = 0u;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const float4 b4 = *reinterpret_cast<const float4*>(sBias + l * 128 + c0 + 4 * q);
          v[4 * q] = __uint_as_float(r[4 * q]) + b4.x;
          v[4 * q + 1] = __uint_as_float(r[4 * q + 1]) + b4.y;
          v[4 * q + 2] = __uint_as_float(r[4 * q + 2]) + b4.z;
          v[4 * q + 3] = __uint_as_float(r[4 * q + 3]) + b4.w;
        }
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          const bool pos = v[i] > 0.f;
          bits |= (pos ? 1u : 0u) << i;
          v[i] = pos ? v[i] : neg_slope * v[i];
        }
        mask[l][gi_] = bits;
        uint32_t w[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) w[i] = pack_f16(v[2 * i], v[2 * i + 1]);
        tmem_st8(tA + lane_off + (uint32_t)(c0 >> 1), w);
        if (l == t - 1) store_row16(sH, c0, w);
      });
      publish(l == t - 1);
    }
    TL(1);
    // ---- heads: outputs, then delta of the four head pre-activations (scaled) ---------------------------
    if (warp == 0) {
      const uint32_t issue = elect_one();
      const uint32_t idesc = make_idesc(16, false, false);
      for (int ks = 0; ks < net.head_in / 16; ++ks)
        umma_ts(tD, tA + ks * 8, make_desc(sW_addr + L * kTileBytes + (ks >> 2) * 2048 + (ks & 3) * 32, 16, 1024), idesc,
                ks > 0, issue);
      umma_commit_if(bar, issue);
    }
    wait_mma();
    if (half == 0) {
      float v[16];
      tmem_ld16(tD + lane_off, v);
      float dh[4];
      const float gs[3] = {go.x * scale, go.y * scale, go.z * scale};
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const float y = 1.f / (1.f + __expf(-(v[c] + sBias[L * 128 + c])));
        dh[c] = gs[c] * y * (1.f - y);
      }
      dh[3] = (v[3] + sBias[L * 128 + 3]) > 0.f ? go.w * scale : 0.f;
      uint32_t w[8] = {pack_f16(dh[0], dh[1]), pack_f16(dh[2], dh[3]), 0u, 0u, 0u, 0u, 0u, 0u};
      tmem_st8(tAH + lane_off, w);
      if (t == L) *reinterpret_cast<uint4*>(sDelta + tile_off(row, 0, 16384)) = make_uint4(w[0], w[1], 0u, 0u);
    }
    TL(2);
    // ---- delta recursion down to the target layer ---------------------------------------------------------
    if (t < L) {
      publish(false);
      if (warp == 0) {   // G_{L-1} = delta_head W_head: K = the 16 rows of the head tile, read MN-major
        const uint32_t issue = elect_one();
        umma_ts(tD, tAH, make_desc(sW_addr + L * kTileBytes, 2048, 1024), make_idesc(net.head_in, false, true), 0u, issue);
        umma_commit_if(bar, issue);
      }
      wait_mma();
      for (int l = L - 1; l >= t; --l) {
        const int nl = net.out[l];
        for_groups(tD + lane_off, 16 * half, nl, [&](const uint32_t* r, int c0, int gi_) {
          uint32_t bits = 0u;
#pragma unroll
          for (int ll = 0; ll < 4; ++ll)
            if (ll == l) bits = mask[ll][gi_];
          uint32_t w[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const float lo = __uint_as_float(r[2 * i]), hi = __uint_as_float(r[2 * i + 1]);
            w[i] = pack_f16(((bits >> (2 * i)) & 1u) ? lo : neg_slope * lo, ((bits >> (2 * i + 1)) & 1u) ? hi : neg_slope * hi);
          }
          if (l == t) store_row16(sDelta, c0, w);
          if (l != t || (t == 0 && want_x)) tmem_st8(tA + lane_off + (uint32_t)(c0 >> 1), w);   // delta_0 also feeds dL/dx
        });
        if (l == t) break;
        publish(false);
        if (warp == 0) {   // G_{l-1} = delta_l W_l: B[n][k] = W_l[k][n], the forward tile read MN-major
          const uint32_t issue = elect_one();
          const uint32_t idesc = make_idesc(net.in[l], false, true);
          for (int ks = 0; ks < nl / 16; ++ks)
            umma_ts(tD, tA + ks * 8, make_desc(sW_addr + l * kTileBytes + ks * 2048, 16384, 1024), idesc, ks > 0, issue);
          umma_commit_if(bar, issue);
        }
        wait_mma();
      }
    }
    TL(3);
    // ---- dW_t += delta_t^T h_{t-1}: K = the 128 rows of the tile, both operands MN-major ---------------------
    publish(true);
    if (warp == 0) {
      const uint32_t issue = elect_one();
      const uint32_t idesc = make_idesc(k_t, true, true);
      for (int ks = 0; ks < kRowsT / 16; ++ks)
        umma_ss(tDW, make_desc(sDelta_addr + ks * 2048, 16384, 1024), make_desc(sH_addr + ks * 2048, 16384, 1024), idesc,
                (tiles_done > 0 || ks > 0) ? 1u : 0u, issue);
      if (t == 0 && want_x) {   // a1: dL/dx = delta_0 W_0 (the layer-0 tile read MN-major), into the free accumulator
        const uint32_t idx_ = make_idesc(net.k0_pad, false, true);
        for (int ks = 0; ks < net.out[0] / 16; ++ks)
          umma_ts(tD, tA + ks * 8, make_desc(sW_addr + ks * 2048, 16384, 1024), idx_, ks > 0, issue);
      }
      umma_commit_if(bar, issue);
    }
    {   // db_t[f] += sum over the rows of delta_t[row][f], f = tid (read while the MMAs run)
      float s = 0.f;
      for (int r = 64 * half; r < 64 * half + 64; ++r) s += __half2float(*reinterpret_cast<const __half*>(sDelta + tile_off(r, row, 16384)));
      db += s;
    }
    wait_mma();   // the operand tiles are free again
    if (t == 0 && want_x) {   // dL/dx of this thread's column groups, through the input assembly to the Gaussian
      for_groups(tD + lane_off, 16 * half, net.k0_pad, [&](const uint32_t* r, int c0, int) {
        if (gi >= 0 && c0 < net.in_dim) {
          float v[16];
#pragma unroll
          for (int k = 0; k < 16; ++k) v[k] = c0 + k < net.in_dim ? __uint_as_float(r[k]) * inv_scale : 0.f;
          input_row_back(a.g, gi, a.cam.pos, a.lights.l[li].pos, c0, min(16, net.in_dim - c0), v, a.ig);
        }
      });
      tc_fence_before();
      __syncthreads();   // every thread has read the accumulator before the next tile's MMAs overwrite it
      tc_fence_after();
    }
    ++tiles_done;
    TL(4);
  }

  // ---- the accumulators leave tensor memory: un-scale, one atomic per weight and CTA -----------------------
  if (tiles_done > 0) {
    const int m = row;   // output neuron of the target layer
    int w_row = -1, b_at = -1, n_in = 0;
    if (t < L) {
      if (m < net.out[t]) { w_row = net.w[t] + m * net.in[t]; b_at = net.b[t] + m; }
      n_in = net.in[t];
    } else {
      if (m < 3) { w_row = net.sss_w + m * net.head_in; b_at = net.sss_b + m; }
      else if (m == 3) { w_row = net.inc_w; b_at = net.inc_b; }
      n_in = net.head_in;
    }
    for (int c0 = 16 * half; c0 < k_t; c0 += 32) {
      float v[16];
      tmem_ld16(tDW + lane_off + c0, v);
      if (w_row >= 0) {
#pragma unroll
        for (int i = 0; i < 16; ++i)
          if (c0 + i < n_in && v[i] != 0.f) atomicAdd(&a.g_params[w_row + c0 + i], v[i] * inv_scale);
      }
    }
    if (b_at >= 0 && db != 0.f) atomicAdd(&a.g_params[b_at], db * inv_scale);
  }
#ifdef SSSGS_BWD_TIMELINE
  TL(5);
  if (tid == 0 && blockIdx.x == 0)
    printf("target %d tiles %u: x %lld fwd %lld head %lld rec %lld dW %lld out %lld | before-wait %lld in-wait %lld (clk per tile)\n", t, tiles_done,
           tl[0] / max(tiles_done, 1u), tl[1] / max(tiles_done, 1u), tl[2] / max(tiles_done, 1u), tl[3] / max(tiles_done, 1u),
           tl[4] / max(tiles_done, 1u), tl[5], tl[6] / max(tiles_done, 1u), tl[7] / max(tiles_done, 1u));
#endif
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
}

}  // namespace tc

// ---- a3 backward: dL/d(2-D mean, conic, depth) -> dL/d(mean, scale, rotation) -------------------------------
// Reverse mode of the EWA projection (Eq. 2), per Gaussian, hand derived:
//   p = R mu + t, (u, w) = (p_x, p_y) / z, pix = (fx u + cx, fy w + cy), depth = z,
//   J = [[fx/z, 0, -fx u_cl/z], [0, fy/z, -fy w_cl/z]] (u_cl, w_cl: frustum clamp, constant where it clamps),
//   T = J R, Sigma = M M^T with M = Rq diag(s), (a, b, c) = T Sigma T^T + 0.3 I, conic = (c, -b, a) / (a c - b^2).
// Plain fp32 (the canonical rounding sequence of project_kernel only matters for keys); Gaussians without an
// upstream gradient (culled, never blended) get zeros.
__global__ void __launch_bounds__(256)
project_backward_kernel(int64_t n, const float* __restrict__ means, const float* __restrict__ scales,
                        const float* __restrict__ rotations, CamParams cam, const float* __restrict__ g_mean2d,
                        const float* __restrict__ g_conic, const float* __restrict__ g_depth,
                        float* __restrict__ d_means, float* __restrict__ d_scales, float* __restrict__ d_rot) {
  const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (i >= n) return;
  const float gpx = g_mean2d[2 * i], gpy = g_mean2d[2 * i + 1];
  const float gca = g_conic[3 * i], gcb = g_conic[3 * i + 1], gcc = g_conic[3 * i + 2];
  const float gz = g_depth[i];
  float dmu[3] = {0.f, 0.f, 0.f}, ds[3] = {0.f, 0.f, 0.f}, dq[4] = {0.f, 0.f, 0.f, 0.f};
  if (gpx != 0.f || gpy != 0.f || gca != 0.f || gcb != 0.f || gcc != 0.f || gz != 0.f) {
    const float* R = cam.R;
    const float mu[3] = {means[3 * i], means[3 * i + 1], means[3 * i + 2]};
    float p[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) p[k] = R[3 * k] * mu[0] + R[3 * k + 1] * mu[1] + R[3 * k + 2] * mu[2] + cam.t[k];
    const float z = p[2], iz = 1.f / z;
    const float u = p[0] * iz, w = p[1] * iz;
    const float lx = kFrustumClamp * cam.tanx, ly = kFrustumClamp * cam.tany;
    const bool free_x = u > -lx && u < lx, free_y = w > -ly && w < ly;
    const float ucl = fminf(lx, fmaxf(-lx, u)), wcl = fminf(ly, fmaxf(-ly, w));
    const float j00 = cam.fx * iz, j11 = cam.fy * iz, j02 = -cam.fx * ucl * iz, j12 = -cam.fy * wcl * iz;
    float T0[3], T1[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      T0[k] = j00 * R[k] + j02 * R[6 + k];
      T1[k] = j11 * R[3 + k] + j12 * R[6 + k];
    }
    const float qr = rotations[4 * i], qx = rotations[4 * i + 1], qy = rotations[4 * i + 2], qz = rotations[4 * i + 3];
    const float sc[3] = {scales[3 * i], scales[3 * i + 1], scales[3 * i + 2]};
    float Rq[9];
    Rq[0] = 1.f - 2.f * (qy * qy + qz * qz); Rq[1] = 2.f * (qx * qy - qr * qz); Rq[2] = 2.f * (qx * qz + qr * qy);
    Rq[3] = 2.f * (qx * qy + qr * qz); Rq[4] = 1.f - 2.f * (qx * qx + qz * qz); Rq[5] = 2.f * (qy * qz - qr * qx);
    Rq[6] = 2.f * (qx * qz - qr * qy); Rq[7] = 2.f * (qy * qz + qr * qx); Rq[8] = 1.f - 2.f * (qx * qx + qy * qy);
    float M[9], Sg[9];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) M[3 * a + b] = Rq[3 * a + b] * sc[b];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) Sg[3 * a + b] = M[3 * a] * M[3 * b] + M[3 * a + 1] * M[3 * b + 1] + M[3 * a + 2] * M[3 * b + 2];
    float S0[3], S1[3];   // Sigma T0, Sigma T1
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      S0[k] = Sg[3 * k] * T0[0] + Sg[3 * k + 1] * T0[1] + Sg[3 * k + 2] * T0[2];
      S1[k] = Sg[3 * k] * T1[0] + Sg[3 * k + 1] * T1[1] + Sg[3 * k + 2] * T1[2];
    }
    const float a = dot3f(T0, S0) + kLowPass, b = dot3f(T1, S0), c = dot3f(T1, S1) + kLowPass;
    const float det = a * c - b * b;
    if (det > 0.f && z > 0.f) {
      // conic = (c, -b, a) / det
      const float id = 1.f / det;
      const float common = (gca * c - gcb * b + gcc * a) * id * id;
      const float da = gcc * id - common * c;
      const float dc = gca * id - common * a;
      const float db = -gcb * id + common * 2.f * b;
      // (a, b, c) -> T0, T1, Sigma
      float dT0[3], dT1[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        dT0[k] = 2.f * da * S0[k] + db * S1[k];
        dT1[k] = 2.f * dc * S1[k] + db * S0[k];
      }
      float dM[9];   // dM = (dSigma + dSigma^T) M, dSigma_ij = da T0_i T0_j + db T1_i T0_j + dc T1_i T1_j
#pragma unroll
      for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int col = 0; col < 3; ++col) {
          float acc = 0.f;
#pragma unroll
          for (int k = 0; k < 3; ++k) {
            const float dsym = 2.f * da * T0[r] * T0[k] + db * (T1[r] * T0[k] + T0[r] * T1[k]) + 2.f * dc * T1[r] * T1[k];
            acc += dsym * M[3 * k + col];
          }
          dM[3 * r + col] = acc;
        }
      float dRq[9];
#pragma unroll
      for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int col = 0; col < 3; ++col) {
          dRq[3 * r + col] = dM[3 * r + col] * sc[col];
          ds[col] += dM[3 * r + col] * Rq[3 * r + col];
        }
      dq[0] = 2.f * (-qz * dRq[1] + qy * dRq[2] + qz * dRq[3] - qx * dRq[5] - qy * dRq[6] + qx * dRq[7]);
      dq[1] = 2.f * (qy * dRq[1] + qz * dRq[2] + qy * dRq[3] - 2.f * qx * dRq[4] - qr * dRq[5] + qz * dRq[6] + qr * dRq[7] - 2.f * qx * dRq[8]);
      dq[2] = 2.f * (-2.f * qy * dRq[0] + qx * dRq[1] + qr * dRq[2] + qx * dRq[3] + qz * dRq[5] - qr * dRq[6] + qz * dRq[7] - 2.f * qy * dRq[8]);
      dq[3] = 2.f * (-2.f * qz * dRq[0] - qr * dRq[1] + qx * dRq[2] + qr * dRq[3] - 2.f * qz * dRq[4] + qy * dRq[5] + qx * dRq[6] + qy * dRq[7]);
      // T -> J entries -> (u, w, z)
      const float dj00 = dT0[0] * R[0] + dT0[1] * R[1] + dT0[2] * R[2];
      const float dj02 = dT0[0] * R[6] + dT0[1] * R[7] + dT0[2] * R[8];
      const float dj11 = dT1[0] * R[3] + dT1[1] * R[4] + dT1[2] * R[5];
      const float dj12 = dT1[0] * R[6] + dT1[1] * R[7] + dT1[2] * R[8];
      float du = cam.fx * gpx, dw = cam.fy * gpy, dz = gz;
      dz += -cam.fx * iz * iz * dj00 - cam.fy * iz * iz * dj11 + cam.fx * ucl * iz * iz * dj02 + cam.fy * wcl * iz * iz * dj12;
      if (free_x) du += -cam.fx * iz * dj02;
      if (free_y) dw += -cam.fy * iz * dj12;
      // (u, w) = (p_x, p_y) / z
      const float dp[3] = {du * iz, dw * iz, dz - (u * du + w * dw) * iz};
#pragma unroll
      for (int k = 0; k < 3; ++k) dmu[k] = R[k] * dp[0] + R[3 + k] * dp[1] + R[6 + k] * dp[2];
    }
  }
  // added to what the a1 backward may have accumulated (the arrays start from zero)
#pragma unroll
  for (int k = 0; k < 3; ++k) { d_means[3 * i + k] += dmu[k]; d_scales[3 * i + k] += ds[k]; }
#pragma unroll
  for (int k = 0; k < 4; ++k) d_rot[4 * i + k] += dq[k];
}

__global__ void __launch_bounds__(256) zero_kernel(float* p, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)gridDim.x * 256) p[i] = 0.f;
}

}  // namespace

int launch_zero(float* p, int64_t n, cudaStream_t s) {
  if (!p || n <= 0) return 0;
  int64_t blocks = (n + 255) / 256;
  if (blocks > 148 * 8) blocks = 148 * 8;
  zero_kernel<<<(unsigned)blocks, 256, 0, s>>>(p, n);
  return 1;
}

int launch_project_backward(const sssgs_gaussians& g, const CamParams& cam, const float* g_mean2d, const float* g_conic,
                            const float* g_depth, float* d_means, float* d_scales, float* d_rot, cudaStream_t s) {
  if (g.n == 0) return 0;
  project_backward_kernel<<<(unsigned)((g.n + 255) / 256), 256, 0, s>>>(g.n, g.means, g.scales, g.rotations, cam, g_mean2d,
                                                                       g_conic, g_depth, d_means, d_scales, d_rot);
  return 1;
}

int launch_shade_backward(const CamParams& cam, const LightBatch& lights, int n_lights, const float* gbuf,
                          const float* grad_rgb, const float* grad_gbuf_in, float* grad_gbuf, cudaStream_t s) {
  const int64_t npix = (int64_t)cam.width * cam.height;
  const int64_t total = npix * n_lights;
  if (total == 0) return 0;
  shade_backward_kernel<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(cam, lights, n_lights, npix, gbuf, grad_rgb, grad_gbuf_in, grad_gbuf);
  return 1;
}

int launch_composite_backward(const CamParams& cam, int n_lights, const GeomBuffers& gb, const uint32_t* sorted_vals,
                              const float4* attr, const float4* mlp_out, int mlp_stride, const float* grad_gbuf,
                              float* g_opacity, float* g_mean2d, float* g_conic, float* g_depth, float* g_attr,
                              float* g_mlp_out, int64_t n, cudaStream_t s) {
  const int tiles = cam.tiles_x * cam.tiles_y;
  if (tiles == 0 || n_lights == 0) return 0;
  const int64_t npix = (int64_t)cam.width * cam.height;
#define SSSGS_CB(LB)                                                                                              \
  composite_backward_kernel<LB><<<tiles, 256, 0, s>>>(cam, n_lights, gb.ranges, gb.tile_order, sorted_vals, gb.rec_a, gb.rec_b, attr, \
                                                      mlp_out, mlp_stride, grad_gbuf, npix, g_opacity, g_mean2d,   \
                                                      g_conic, g_depth, g_attr, g_mlp_out, n)
  if (n_lights <= 1) SSSGS_CB(1);
  else if (n_lights <= 4) SSSGS_CB(4);
  else SSSGS_CB(8);
#undef SSSGS_CB
  return 1;
}

int launch_mlp_backward(const sssgs_gaussians& g, const sssgs_mlp& mlp, const CamParams& cam, const LightBatch& lights,
                        int n_lights, const float* g_mlp_out, float* g_params, uint32_t* row_list, uint32_t* row_count,
                        uint8_t* blob, bool pack, bool force_fp32, float* const input_grads[6], int num_sms, cudaStream_t s) {
  if (g.n == 0 || n_lights == 0 || !g_params) return 0;
  InputGrads ig;   // means, scales, rotations, attr, feat, vis_sh
  ig.means = input_grads[0]; ig.scales = input_grads[1]; ig.rotations = input_grads[2]; ig.attr = input_grads[3];
  ig.feat = input_grads[4]; ig.vis_sh = input_grads[5];
  int launches = 0;
  const int64_t rows = g.n * n_lights;
  if (cudaMemsetAsync(row_count, 0, 8, s) != cudaSuccess) return 0;
  int64_t cb = (rows + 255) / 256;
  if (cb > (int64_t)num_sms * 8) cb = (int64_t)num_sms * 8;
  bwd_rows_kernel<<<(unsigned)cb, 256, 0, s>>>(reinterpret_cast<const float4*>(g_mlp_out), rows, row_list, row_count);
  ++launches;

  // ---- tensor-core path: a chain of <= 4 trunk layers and the two heads -------------------------------------
  // The tensor-core path re-evaluates the forward pass with binary16 operands: it only matches a forward pass that
  // ran with binary16 operands too.  A bf16 forward (sssgs_mlp.compute) is differentiated on the fp32 path.
  bool use_tc = !force_fp32 && mlp.compute == SSSGS_COMPUTE_FP16 && mlp.n_inc_hidden == 0 && mlp.n_trunk >= 1 &&
                mlp.n_trunk <= 4 && mlp.in_dim <= 128;
  for (int l = 0; l < mlp.n_trunk && use_tc; ++l)
    use_tc = mlp.trunk_width[l] % 16 == 0 && mlp.trunk_width[l] >= 16 && mlp.trunk_width[l] <= 128;
  if (use_tc) {
    tc::TcNet net;
    memset(&net, 0, sizeof net);
    net.n_trunk = mlp.n_trunk;
    net.in_dim = mlp.in_dim;
    net.k0_pad = (mlp.in_dim + 15) & ~15;
    net.activation = mlp.activation;
    net.slope = mlp.leaky_slope;
    int off = 0, d = mlp.in_dim;
    for (int l = 0; l < mlp.n_trunk; ++l) {
      const int o = mlp.trunk_width[l];
      net.out[l] = o; net.in[l] = d; net.w[l] = off; net.b[l] = off + o * d;
      off += o * d + o;
      d = o;
    }
    net.head_in = d;
    net.sss_w = off; net.sss_b = off + 3 * d;
    off += 3 * d + 3;
    net.inc_w = off; net.inc_b = off + d;
    if (pack) {
      tc::bwd_pack_kernel<<<64, 256, 0, s>>>(net, (const float*)mlp.params, blob);
      ++launches;
    }
    const int smem = tc::tc_smem_bytes(net.n_trunk);
    if (ensure_dyn_smem((const void*)tc::mlp_backward_tc_kernel, smem) != cudaSuccess) return launches;
    tc::TcArgs a;
    a.g = g; a.net = net; a.cam = cam; a.lights = lights; a.n = g.n;
    a.list = row_list; a.count = row_count; a.gomax_bits = row_count + 1;
    a.g_mlp_out = g_mlp_out; a.blob = blob; a.g_params = g_params; a.ig = ig;
    int gx = num_sms / (net.n_trunk + 1);
    if (gx < 1) gx = 1;
    tc::mlp_backward_tc_kernel<<<dim3((unsigned)gx, (unsigned)(net.n_trunk + 1)), 256, smem, s>>>(a);
    return launches + 1;
  }

  // ---- fp32 CUDA-core path ------------------------------------------------------------------------------------
  BwdNet net;
  net.in_dim = mlp.in_dim;
  net.activation = mlp.activation;
  net.slope = mlp.leaky_slope;
  int off = 0, d = mlp.in_dim, nl = 0;
  for (int l = 0; l < mlp.n_trunk; ++l) {
    const int o = mlp.trunk_width[l];
    net.L[nl] = BwdLayer{off, off + o * d, o, d, nl - 1, K_HIDDEN};
    off += o * d + o;
    d = o;
    ++nl;
  }
  const int trunk_last = nl - 1;
  net.trunk_last = trunk_last;
  net.L[nl] = BwdLayer{off, off + 3 * d, 3, d, trunk_last, K_SSS};
  off += 3 * d + 3;
  ++nl;
  int src = trunk_last, di = d;
  for (int l = 0; l < mlp.n_inc_hidden; ++l) {
    const int o = mlp.inc_hidden_width[l];
    net.L[nl] = BwdLayer{off, off + o * di, o, di, src, K_HIDDEN};
    off += o * di + o;
    src = nl;
    di = o;
    ++nl;
  }
  net.L[nl] = BwdLayer{off, off + di, 1, di, src, K_INC_OUT};
  ++nl;
  net.n_layers = nl;
  const int smem = (128 * kWS + 3 * kBR * 128 + kBR * 4 + (nl + 1) * kBR * 128) * 4;
  if (ensure_dyn_smem((const void*)mlp_backward_kernel, smem) != cudaSuccess) return launches;
  int gx = num_sms / nl;
  if (gx < 1) gx = 1;
  mlp_backward_kernel<<<dim3((unsigned)gx, (unsigned)nl), 256, smem, s>>>(g, net, (const float*)mlp.params, cam, lights, g.n,
                                                                        row_list, row_count, g_mlp_out, g_params, ig);
  return launches + 1;
}

}  // namespace sssgs

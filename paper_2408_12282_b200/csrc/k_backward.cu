// Backward pass of hot-path steps a8 (deferred shading), a7 (compositing) and a2 (the MLP)
// ("optimize all parameters jointly via raytraced differentiable rendering",
// L112, L343-349: the losses are functions of the rendered image and of the rasterised property images).
//
// For one camera and its lights, with G_l = dL / d rgb_l given by the caller (L = sum_l <G_l, rgb_l>):
//   shade_backward_kernel      per (light, pixel): dL / d gbuffer_l[p][0..15]           (Eq. 4, Eq. 7)
//   composite_backward_kernel  per tile, walking its list back to front: dL / d (opacity, 2-D mean, conic,
//                              depth, normal, base colour, roughness, metalness, sss) per Gaussian and
//                              dL / d (L_SSS, L_in) per (Gaussian, light)                        (Eq. 3)
//   mlp_backward_*             dL / d Theta (weights and biases of every layer)             (Eq. 6)
// The discontinuous decisions of the forward pass (alpha >= 1/255, power <= 0, the T' < 1e-4 stop, the 0.99
// clamp, the ReLUs) are constants of the differentiation.  Arithmetic is fp32 throughout; the MLP is
// re-evaluated in fp32 from the caller's parameters (this first version runs on the CUDA cores: the
// tensor-core forward keeps no activations, DESIGN.md section 7e says what a tcgen05 version needs).
// Per-Gaussian sums are formed with float atomics: results are reproducible to rounding, not bit for bit.
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
                      float* __restrict__ grad_gbuf) {
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
composite_backward_kernel(CamParams cam, int n_lights, const uint2* __restrict__ ranges,
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
  const int tile = blockIdx.x;
  const int tx = tile % cam.tiles_x, ty = tile / cam.tiles_x;
  const int px = tx * kTile + (warp & 1) * 8 + (lane & 7), py = ty * kTile + (warp >> 1) * 4 + (lane >> 3);
  const bool inside = px < cam.width && py < cam.height;
  const int64_t pidx = (int64_t)min(py, cam.height - 1) * cam.width + min(px, cam.width - 1);
  const uint2 range = ranges[tile];
  const int n_entries = (int)(range.y - range.x);
  constexpr float kInvLog2e = 0.6931471805599453f;   // rec_b holds the conic scaled by -log2(e)/2, -log2(e), -log2(e)/2
  // upstream gradients of this pixel: light-independent channels summed over the lights, MLP channels per light
  float dGs[11];   // depth, n3, b3, rough, metal, sss, A
  float dGl[LB][4];
  for (int c = 0; c < 11; ++c) dGs[c] = 0.f;
  for (int l = 0; l < LB; ++l)
    for (int c = 0; c < 4; ++c) dGl[l][c] = 0.f;
  if (inside) {
    for (int l = 0; l < LB; ++l) {
      if (l >= n_lights) break;
      const float* gp = grad_gbuf + ((int64_t)l * npix + pidx) * 16;
      for (int c = 0; c < 10; ++c) dGs[c] += gp[c];
      dGs[10] += gp[14];
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
    for (int j = 0; j < cnt && !done; ++j) {
      const float4 ra = s_a[j], rb = s_b[j];
      const float dx = (float)px - ra.x, dy = (float)py - ra.y;
      const float p2 = fmaf(fmaf(rb.y, dy, rb.x * dx), dx, rb.z * dy * dy);   // log2(e) * power, as in the forward walk
      float al;
      asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(al) : "f"(p2));
      al = fminf(kAlphaMax, rb.w * al);
      if (p2 <= 0.f && al >= kAlphaMin) {
        const float Tn = T * (1.f - al);
        if (Tn < kTMin) { done = true; break; }
        T = Tn;
        last = b0 + j + 1;
      }
    }
  }
  atomicMax(&s_last, last);
  __syncthreads();
  const int max_last = s_last;
  // ---- phase B: back to front ---------------------------------------------------------------------
  float R = 0.f;   // sum_{j > i} w_j Phi_j
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
    for (int j = cnt - 1; j >= 0; --j) {
      const float4 ra = s_a[j], rb = s_b[j];
      const uint32_t gid = s_g[j];
      const float dx = (float)px - ra.x, dy = (float)py - ra.y;
      const float p2 = fmaf(fmaf(rb.y, dy, rb.x * dx), dx, rb.z * dy * dy);
      float e;
      asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(p2));
      const float araw = rb.w * e;
      const float al = fminf(kAlphaMax, araw);
      const bool blended = inside && (b0 + j) < last && p2 <= 0.f && al >= kAlphaMin;
      float w = 0.f, d_alpha = 0.f;
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
      if (__any_sync(0xFFFFFFFFu, blended)) {
        // alpha = o e^power (unclamped); power = -(a dx^2 + c dy^2) / 2 - b dx dy
        const bool unclamped = araw < kAlphaMax;
        const float d_o = (blended && unclamped) ? d_alpha * e : 0.f;
        const float d_pow = (blended && unclamped) ? d_alpha * al : 0.f;
        const float ca = -2.f * kInvLog2e * rb.x, cb = -kInvLog2e * rb.y, cc = -2.f * kInvLog2e * rb.z;
        float vals[6 + 11 + 4 * LB];
        vals[0] = d_o;
        vals[1] = d_pow * (ca * dx + cb * dy);      // d power / d pix_x
        vals[2] = d_pow * (cc * dy + cb * dx);
        vals[3] = d_pow * (-0.5f * dx * dx);         // d power / d conic a, b, c
        vals[4] = d_pow * (-dx * dy);
        vals[5] = d_pow * (-0.5f * dy * dy);
        for (int c = 0; c < 10; ++c) vals[6 + c] = w * dGs[c];
        vals[16] = 0.f;
        for (int l = 0; l < LB; ++l)
          for (int c = 0; c < 4; ++c) vals[17 + 4 * l + c] = w * dGl[l][c];
#pragma unroll
        for (int q = 0; q < 6 + 11 + 4 * LB; ++q) {
          float s = vals[q];
#pragma unroll
          for (int o = 16; o >= 1; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
          vals[q] = s;
        }
        if (lane == 0) {
          atomicAdd(&g_opacity[gid], vals[0]);
          atomicAdd(&g_mean2d[2 * (size_t)gid], vals[1]);
          atomicAdd(&g_mean2d[2 * (size_t)gid + 1], vals[2]);
          atomicAdd(&g_conic[3 * (size_t)gid], vals[3]);
          atomicAdd(&g_conic[3 * (size_t)gid + 1], vals[4]);
          atomicAdd(&g_conic[3 * (size_t)gid + 2], vals[5]);
          atomicAdd(&g_depth[gid], vals[6]);
          // g_attr: [n][9] = normal (3), base colour (3), roughness, metalness, sss
          for (int c = 0; c < 9; ++c) atomicAdd(&g_attr[9 * (size_t)gid + c], vals[7 + c]);
          for (int l = 0; l < LB; ++l) {
            if (l >= n_lights) break;
            for (int c = 0; c < 4; ++c) atomicAdd(&g_mlp_out[((size_t)l * n + gid) * 4 + c], vals[17 + 4 * l + c]);
          }
        }
      }
    }
  }
}

// ---- a2 backward (fp32, CUDA cores) ----------------------------------------------------------------
// The MLP input row of (Gaussian, light), as the forward kernel assembles it.
__device__ __forceinline__ void mlp_input_row(const sssgs_gaussians& g, int64_t i, const float* cam_pos,
                                              const float* light_pos, float* x) {
  const float mu[3] = {g.means[3 * i], g.means[3 * i + 1], g.means[3 * i + 2]};
  for (int k = 0; k < 3; ++k) x[k] = g.normals[3 * i + k];
  const float sgn = g.rotations[4 * i] < 0.f ? -1.f : 1.f;
  x[3] = sgn * g.rotations[4 * i];
  x[4] = sgn * g.rotations[4 * i + 1];
  for (int k = 0; k < 3; ++k) x[5 + k] = g.scales[3 * i + k];
  float wi[3], wo[3];
  for (int k = 0; k < 3; ++k) { wi[k] = light_pos[k] - mu[k]; wo[k] = cam_pos[k] - mu[k]; }
  const float d = sqrtf(dot3f(wi, wi)), dn = sqrtf(dot3f(wo, wo));
  for (int k = 0; k < 3; ++k) { x[8 + k] = wi[k] / d; x[11 + k] = wo[k] / dn; }
  x[14] = d;
  const int nc = (g.vis_sh_degree + 1) * (g.vis_sh_degree + 1);
  float v = 0.2820948f * g.vis_sh[nc * i];
  if (g.vis_sh_degree >= 1)
    v += 0.4886025f * (g.vis_sh[nc * i + 1] * x[9] + g.vis_sh[nc * i + 2] * x[10] + g.vis_sh[nc * i + 3] * x[8]);
  x[15] = fminf(1.f, fmaxf(0.f, v));
  for (int k = 0; k < 4; ++k)
    for (int a = 0; a < 3; ++a) {
      float s, c;
      sincospif((float)(1 << k) * mu[a], &s, &c);
      x[16 + 6 * k + a] = s;
      x[16 + 6 * k + 3 + a] = c;
    }
  for (int k = 0; k < g.feat_dim; ++k) x[40 + k] = g.feat[(int64_t)g.feat_dim * i + k];
}

// Layer table of the MLP in the caller's parameter packing (sssgs_mlp.params, fp32).
struct BwdLayer { int w, b, out, in, src, kind; };   // src: index of the layer whose output feeds this one (-1: x)
struct BwdNet {
  int n_layers, in_dim, activation;
  float slope;
  BwdLayer L[SSSGS_MAX_TRUNK + SSSGS_MAX_INC_HIDDEN + 2];
};
enum { K_HIDDEN = 0, K_SSS = 1, K_INC_OUT = 2 };
constexpr int kBwdMaxW = 128;
constexpr int kBwdMaxIn = 128;

// One CTA of 128 threads per (Gaussian, light) row, looping over rows; thread t = neuron t.  Activations of
// all layers of the row stay in shared memory; the weight gradients are accumulated straight into global
// memory (atomicAdd of delta_t * h_k: 128 threads sweep the 128 x in matrix of a layer).
__global__ void __launch_bounds__(128)
mlp_backward_kernel(sssgs_gaussians g, BwdNet net, const float* __restrict__ params, CamParams cam, LightBatch lights,
                    int n_lights, int light0, const float* __restrict__ g_mlp_out, int64_t n,
                    float* __restrict__ g_params) {
  __shared__ float s_h[SSSGS_MAX_TRUNK + SSSGS_MAX_INC_HIDDEN + 3][kBwdMaxIn];   // s_h[0] = x, s_h[l + 1] = output of layer l
  __shared__ float s_d[2][kBwdMaxW];
  __shared__ float s_dacc[SSSGS_MAX_TRUNK + SSSGS_MAX_INC_HIDDEN + 3][kBwdMaxW];   // gradient wrt each layer's OUTPUT
  const int t = threadIdx.x;
  (void)s_d;
  for (int64_t row = blockIdx.x; row < n * n_lights; row += gridDim.x) {
    const int64_t i = row % n;
    const int l_idx = (int)(row / n);
    const float* go = g_mlp_out + ((size_t)(light0 + l_idx) * n + i) * 4;
    const float go4[4] = {go[0], go[1], go[2], go[3]};
    if (go4[0] == 0.f && go4[1] == 0.f && go4[2] == 0.f && go4[3] == 0.f) continue;   // row never blended: no gradient
    __syncthreads();
    if (t == 0) mlp_input_row(g, i, cam.pos, lights.l[l_idx].pos, s_h[0]);
    for (int l = 0; l <= net.n_layers; ++l) s_dacc[l][t] = 0.f;
    __syncthreads();
    // ---- forward, fp32 ----
    for (int l = 0; l < net.n_layers; ++l) {
      const BwdLayer& L = net.L[l];
      const float* hin = s_h[L.src + 1];
      if (t < L.out) {
        float s = params[L.b + t];
        const float* W = params + L.w + (size_t)t * L.in;
        for (int k = 0; k < L.in; ++k) s = fmaf(W[k], hin[k], s);
        float y;
        if (L.kind == K_HIDDEN) y = s > 0.f ? s : (net.activation == SSSGS_ACT_LEAKY_RELU ? net.slope * s : 0.f);
        else if (L.kind == K_SSS) y = 1.f / (1.f + expf(-s));
        else y = fmaxf(0.f, s);
        s_h[l + 1][t] = y;
      }
      __syncthreads();
    }
    // ---- backward ----
    for (int l = net.n_layers - 1; l >= 0; --l) {
      const BwdLayer& L = net.L[l];
      // delta_t = dL/d(pre-activation of neuron t of layer l)
      float delta = 0.f;
      if (t < L.out) {
        const float y = s_h[l + 1][t];
        if (L.kind == K_SSS) delta = go4[t] * y * (1.f - y);
        else if (L.kind == K_INC_OUT) delta = y > 0.f ? go4[3] : 0.f;
        else delta = s_dacc[l + 1][t] * (y > 0.f ? 1.f : (net.activation == SSSGS_ACT_LEAKY_RELU ? net.slope : 0.f));
      }
      __syncthreads();
      s_d[0][t] = delta;
      __syncthreads();
      const float* hin = s_h[L.src + 1];
      // dW[t'][k] += delta_t' h_k, db[t'] += delta_t'; d hin[k] += sum_t' W[t'][k] delta_t'
      if (t < L.out && delta != 0.f) atomicAdd(&g_params[L.b + t], delta);
      for (int tp = 0; tp < L.out; ++tp) {
        const float dt = s_d[0][tp];
        if (dt == 0.f) continue;
        if (t < L.in) atomicAdd(&g_params[L.w + (size_t)tp * L.in + t], dt * hin[t]);
      }
      if (L.src >= 0 && t < L.in) {
        float s = 0.f;
        for (int tp = 0; tp < L.out; ++tp) s = fmaf(params[L.w + (size_t)tp * L.in + t], s_d[0][tp], s);
        s_dacc[L.src + 1][t] += s;
      }
      __syncthreads();
    }
  }
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

int launch_shade_backward(const CamParams& cam, const LightBatch& lights, int n_lights, const float* gbuf,
                          const float* grad_rgb, float* grad_gbuf, cudaStream_t s) {
  const int64_t npix = (int64_t)cam.width * cam.height;
  const int64_t total = npix * n_lights;
  if (total == 0) return 0;
  shade_backward_kernel<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(cam, lights, n_lights, npix, gbuf, grad_rgb, grad_gbuf);
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
  composite_backward_kernel<LB><<<tiles, 256, 0, s>>>(cam, n_lights, gb.ranges, sorted_vals, gb.rec_a, gb.rec_b, attr, \
                                                      mlp_out, mlp_stride, grad_gbuf, npix, g_opacity, g_mean2d,   \
                                                      g_conic, g_depth, g_attr, g_mlp_out, n)
  if (n_lights <= 1) SSSGS_CB(1);
  else if (n_lights <= 4) SSSGS_CB(4);
  else SSSGS_CB(8);
#undef SSSGS_CB
  return 1;
}

int launch_mlp_backward(const sssgs_gaussians& g, const sssgs_mlp& mlp, const CamParams& cam, const LightBatch& lights,
                        int n_lights, int light0, const float* g_mlp_out, float* g_params, int num_sms, cudaStream_t s) {
  if (g.n == 0 || n_lights == 0 || !g_params) return 0;
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
  const int64_t rows = g.n * n_lights;
  int64_t blocks = rows < (int64_t)num_sms * 8 ? rows : (int64_t)num_sms * 8;
  mlp_backward_kernel<<<(unsigned)blocks, 128, 0, s>>>(g, net, (const float*)mlp.params, cam, lights, n_lights, light0,
                                                        g_mlp_out, g.n, g_params);
  return 1;
}

}  // namespace sssgs

// Tile rasteriser fused with deferred shading (hot-path steps a7 + a8).
//
// Front-to-back alpha compositing of every property channel (Eq. 3; "we
// accumulate and rasterize each property on the image plane in a deferred shading pipeline",
// L55), then per-pixel shading from the accumulators still in registers (L114): back-project the
// pixel, Cook-Torrance/GGX + diffuse (Eq. 4) times the learned incident light, blended
// with the SSS residual (Eq. 7).  Up to LB lights share one walk of the tile list:
// the compositing weights T_i alpha_i do not depend on the light, only the four MLP channels
// do (OLAT sweeps, L301).
//
// One CTA per 16x16 tile, one thread per pixel (a warp covers an 8x4 pixel block).  List
// entries are staged in shared memory in batches of 128 as component-major float4 arrays
// (gathered with 128-bit loads, all threads sharing the work), and every lane reads them back
// as broadcasts.  Outputs are written once: RGB, and on request the 16-channel G-buffer
// (4 x 128-bit stores per pixel) and the diffuse / specular AOVs (L320).  Nothing else goes
// to HBM: the G-buffer round trip of a separate shading pass is avoided.
#include <cuda_fp16.h>

#include <cstdlib>
#include <cstring>

#include "internal.cuh"

namespace sssgs {

namespace {

constexpr int kBatch = 128;
// stages of the staging ring and its shared-memory footprint, per kernel variant
__host__ __device__ constexpr int raster_stages(int lb, bool mark, bool fwd) { return 4; }  // measured: 3 is slower at 8 lights, 6 costs a resident CTA at 1 light
__host__ __device__ constexpr int raster_comps(int lb, bool mark, bool fwd) { return mark ? 2 : (fwd ? 2 + lb : 5 + lb); }
__host__ __device__ constexpr int raster_smem(int lb, bool mark, bool fwd, int warps) {
  return raster_stages(lb, mark, fwd) * (raster_comps(lb, mark, fwd) * kBatch * 16 + kBatch * 4 + 16) + warps * kBatch + 16;
}
constexpr float kPi = 3.14159265358979323846f;

struct ShadeIn {
  float depth, nx, ny, nz, br, bg, bb, rough, metal, sss;  // already divided by coverage A
};

// Approximate reciprocal / reciprocal square root, one MUFU each (about 1 ulp; the shading tolerance
// is 1e-4).  The operands are floored away from zero and denormals by the caller.
__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
constexpr float kInvPi = 0.31830988618379067154f;

// Eq. 7 with the BRDF of Eq. 4 (L76-80), fp32 restatement of DESIGN.md "Shading",
// split in the part that depends on the shaded point and the view only (ShadeView: shared by all
// lights of a walk) and the part per light (shade_light).
struct ShadeView {
  float xw[3], v[3], n[3];
  bool has_n;           // |n| >= 1e-8: otherwise only the SSS term is shaded
  float nv_k;           // nv (1 - k) + k, nv = max(1e-4, n.v)
  float a2, k, omk;     // alpha^2, k = alpha / 2, 1 - k
  float F0[3], omF0[3]; // Fresnel at normal incidence and its complement
  float fd[3];          // diffuse lobe (1 - metal) base / pi
  float difc;           // (1 - sss) (1 - metal) / pi
  float sss, oms;
};

__device__ __forceinline__ void shade_view(const ShadeIn& q, const float xw[3], const CamParams& cam, ShadeView& s) {
  float vv = 0.f;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    s.xw[k] = xw[k];
    s.v[k] = cam.pos[k] - xw[k];
    vv = fmaf(s.v[k], s.v[k], vv);
  }
  const float iv = rsqrt_approx(vv);
#pragma unroll
  for (int k = 0; k < 3; ++k) s.v[k] *= iv;
  const float nn2 = q.nx * q.nx + q.ny * q.ny + q.nz * q.nz;
  s.has_n = nn2 >= 1e-16f;
  const float in = rsqrt_approx(fmaxf(nn2, 1e-16f));
  s.n[0] = q.nx * in; s.n[1] = q.ny * in; s.n[2] = q.nz * in;
  const float nv = fmaxf(1e-4f, s.n[0] * s.v[0] + s.n[1] * s.v[1] + s.n[2] * s.v[2]);
  const float ar = fmaxf(1e-3f, q.rough * q.rough);
  s.a2 = ar * ar;
  s.k = 0.5f * ar;
  s.omk = 1.f - s.k;
  s.nv_k = fmaf(nv, s.omk, s.k);
  const float base[3] = {q.br, q.bg, q.bb};
  const float omm = 1.f - q.metal;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    s.F0[c] = 0.04f * omm + base[c] * q.metal;
    s.omF0[c] = 1.f - s.F0[c];
    s.fd[c] = omm * base[c] * kInvPi;
  }
  s.sss = q.sss;
  s.oms = 1.f - q.sss;
  s.difc = s.oms * omm * kInvPi;
}

// rgb = intensity * A * L_out (+ (1 - A) bg) for one light; dif / spc are the AOVs of L320.
__device__ __forceinline__ void shade_light(const ShadeView& s, const float lsss[3], float lin, float A,
                                            const CamParams& cam, const LightParams& lt, float rgb[3],
                                            float dif[3], float spc[3], bool with_bg) {
  float brdf[3] = {0.f, 0.f, 0.f};
#pragma unroll
  for (int c = 0; c < 3; ++c) dif[c] = spc[c] = 0.f;
  if (s.has_n) {
    float l[3], ll = 0.f;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      l[k] = lt.pos[k] - s.xw[k];
      ll = fmaf(l[k], l[k], ll);
    }
    const float il = rsqrt_approx(ll);
#pragma unroll
    for (int k = 0; k < 3; ++k) l[k] *= il;
    float h[3] = {l[0] + s.v[0], l[1] + s.v[1], l[2] + s.v[2]};
    const float hl2 = h[0] * h[0] + h[1] * h[1] + h[2] * h[2];
    const bool has_h = hl2 >= 1e-16f;
    const float ih = rsqrt_approx(fmaxf(hl2, 1e-16f));
#pragma unroll
    for (int k = 0; k < 3; ++k) h[k] = has_h ? h[k] * ih : s.n[k];
    const float* n = s.n;
    const float nl = fmaxf(0.f, n[0] * l[0] + n[1] * l[1] + n[2] * l[2]);
    const float nh = __saturatef(n[0] * h[0] + n[1] * h[1] + n[2] * h[2]);
    const float vh = __saturatef(s.v[0] * h[0] + s.v[1] * h[1] + s.v[2] * h[2]);
    // cancellation-free GGX: 1 - nh^2 = |n x h|^2
    const float cx = n[1] * h[2] - n[2] * h[1], cy = n[2] * h[0] - n[0] * h[2],
                cz = n[0] * h[1] - n[1] * h[0];
    const float s2 = cx * cx + cy * cy + cz * cz;
    const float dd = fmaxf(1e-12f, s.a2 * nh * nh + s2);  // floor: only n = -h exactly (DESIGN.md readings)
    // D V = a2 / (pi dd^2) / (4 (nl (1 - k) + k) (nv (1 - k) + k))
    const float DV = s.a2 * rcp_approx(kPi * dd * dd * 4.f * fmaf(nl, s.omk, s.k) * s.nv_k);
    const float om = 1.f - vh;
    const float om2 = om * om;
    const float om5 = om2 * om2 * om;
    const float lnl = lin * nl;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float fs = DV * fmaf(s.omF0[c], om5, s.F0[c]);
      brdf[c] = (fs + s.fd[c]) * lnl;
      spc[c] = s.oms * fs * lnl;
      dif[c] = s.difc * lnl;
    }
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const float lout = s.sss * lsss[c] + s.oms * brdf[c];
    rgb[c] = lt.intensity[c] * A * lout + (with_bg ? (1.f - A) * cam.bg[c] : 0.f);
  }
}

__device__ __forceinline__ void shade_point(const ShadeIn& q, const float lsss[3], float lin, float A,
                                            const float xw[3], const CamParams& cam,
                                            const LightParams& lt, float rgb[3], float dif[3],
                                            float spc[3], bool with_bg) {
  ShadeView s;
  shade_view(q, xw, cam, s);
  shade_light(s, lsss, lin, A, cam, lt, rgb, dif, spc, with_bg);
}

// Deferred shading of one pixel (L114): the pixel is projected back to 3-D at its composited depth,
// camera -> world: x = R^T (x_c - t).
__device__ __forceinline__ void backproject(float depth, int px, int py, const CamParams& cam, float xw[3]) {
  const float xc0 = ((float)px - cam.cx) / cam.fx * depth - cam.t[0];
  const float xc1 = ((float)py - cam.cy) / cam.fy * depth - cam.t[1];
  const float xc2 = depth - cam.t[2];
#pragma unroll
  for (int k = 0; k < 3; ++k) xw[k] = cam.R[0 + k] * xc0 + cam.R[3 + k] * xc1 + cam.R[6 + k] * xc2;
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
// 2^x, single MUFU.EX2 (flushes denormal results to zero: alpha is thresholded at 1/255 anyway)
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// Packed fp32x2 arithmetic (sm_100 FFMA2): the walk is bound by instruction issue, and a blend is
// a row of FMAs with one common factor w, so two accumulators ride in one 64-bit register pair.
// Each half is an IEEE fma: results are bit-identical to scalar fmaf.
typedef float2 f32x2;
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) { lo = v.x; hi = v.y; }
// acc += (w, w) * (b0, b1)
__device__ __forceinline__ void fma2(f32x2& acc, f32x2 ww, float b0, float b1) {
  acc = __ffma2_rn(ww, make_float2(b0, b1), acc);
}
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gmem_src) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gmem_src) : "memory");
}
// mbarriers of the staging ring
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(
                   (uint32_t)__cvta_generic_to_shared(bar))
               : "memory");
}
// this thread's arrival happens when all cp.async it has issued so far have landed
__device__ __forceinline__ void mbar_arrive_on_copies(uint64_t* bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"((uint32_t)__cvta_generic_to_shared(bar))
               : "memory");
}
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {  // non-blocking
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
// one try_wait: the hardware may park the thread until the phase completes or a time limit passes
__device__ __forceinline__ bool mbar_try(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(parity)
        : "memory");
  } while (!ok);
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Work decomposition of one rasteriser variant.  A warp covers P = 32/E pixels (a PW x PH block)
// and evaluates E consecutive list entries of that block at once ("entry slots"): lane =
// slot * P + pixel.  A CTA of WARPS warps covers an RW x RH pixel region of a 16x16 tile, so a
// tile is rendered by (16/RW) x (16/RH) CTAs that walk the same list.  E = 1, WARPS = 8 is the
// classic one-thread-per-pixel, one-CTA-per-tile layout; E > 1 shortens the sequential walk of a
// long list by E (more warps share it) and culls at a finer pixel-block granularity.
template <int E, int WARPS>
struct RasterShape {
  static constexpr int P = 32 / E;
  static constexpr int PW = (E == 1) ? 8 : (E == 8 ? 2 : 4);
  static constexpr int PH = P / PW;
  static constexpr int NPIX = WARPS * P;
  static constexpr int RW = NPIX >= 128 ? 16 : 8;
  static constexpr int RH = NPIX / RW;
  static constexpr int SX = kTile / RW, SY = kTile / RH;
  static constexpr int SUBS = SX * SY;
  static constexpr int THREADS = WARPS * 32;
  static_assert(RH >= PH && RH <= kTile && (RW % PW) == 0 && (RH % PH) == 0, "bad raster shape");
};

// End of a pixel's walk, shared by the list walk and the cached walk: unpacks the accumulators, adds
// the E per-slot partial sums of a pixel, writes the G-buffer and shades (L114) -- or, FWD, adds the
// background to the composited per-Gaussian colours.
template <int LB, int E, bool FWD>
__device__ __forceinline__ void raster_finish(float acc_depth, const f32x2* pacc, const f32x2 (*paccl)[2], float A,
                                              float T, bool inside, int px, int py, int slot,
                                              const CamParams& cam, const LightBatch& lights, int n_lights,
                                              float* __restrict__ rgb_out, float* __restrict__ gbuf_out,
                                              float* __restrict__ aovd_out, float* __restrict__ aovs_out,
                                              int64_t frame_stride_px, int sum_mode) {
  constexpr int P = 32 / E;
  constexpr unsigned FULL = 0xFFFFFFFFu;
  // unpack: acc[] in G-buffer channel order (depth, n3, b3, rough, metal, sss), accl[l] = MLP channels
  float acc[10], accl[LB][4];
  acc[0] = acc_depth;
  unpack2(pacc[0], acc[1], acc[2]);
  unpack2(pacc[1], acc[3], acc[7]);
  unpack2(pacc[2], acc[4], acc[5]);
  unpack2(pacc[3], acc[6], acc[8]);
  {
    float a_sum;
    unpack2(pacc[4], acc[9], a_sum);
    if (!FWD) A = a_sum;
  }
#pragma unroll
  for (int l = 0; l < LB; ++l) {
    unpack2(paccl[l][0], accl[l][0], accl[l][1]);
    unpack2(paccl[l][1], accl[l][2], accl[l][3]);
  }

  // ---- combine the E per-slot partial sums of every pixel (all E lanes end up with the total) ----
  if (E > 1) {
#pragma unroll
    for (int o = P; o < 32; o <<= 1) {
#pragma unroll
      for (int c = 0; c < 10; ++c) acc[c] += __shfl_xor_sync(FULL, acc[c], o);
#pragma unroll
      for (int l = 0; l < LB; ++l)
#pragma unroll
        for (int c = 0; c < 4; ++c) accl[l][c] += __shfl_xor_sync(FULL, accl[l][c], o);
      A += __shfl_xor_sync(FULL, A, o);
    }
  }

  if (!inside) return;
  // ---- epilogue: G-buffer stores + deferred shading; lights and store quarters are dealt to the
  //      E lanes of a pixel round-robin ---------------------------------------------------------------
  const int64_t pidx = (int64_t)py * cam.width + px;
  if (FWD) {  // C = sum_i T_i alpha_i c_i + (1 - A) bg  (Eq. 3), lights dealt to the E lanes of a pixel
#pragma unroll
    for (int l = 0; l < LB; ++l) {
      if (l >= n_lights) break;
      if (l % E != slot || !rgb_out) continue;
      float* o = rgb_out + ((int64_t)l * frame_stride_px + pidx) * 3;
#pragma unroll
      for (int c = 0; c < 3; ++c) o[c] = accl[l][c] + (1.f - A) * cam.bg[c];
    }
    return;
  }
  ShadeIn q;
  const bool covered = A >= 1e-6f;
  const float iA = covered ? 1.f / A : 0.f;
  q.depth = acc[0] * iA; q.nx = acc[1] * iA; q.ny = acc[2] * iA; q.nz = acc[3] * iA;
  q.br = acc[4] * iA; q.bg = acc[5] * iA; q.bb = acc[6] * iA;
  q.rough = acc[7] * iA; q.metal = acc[8] * iA; q.sss = acc[9] * iA;
  ShadeView sv;  // light-independent part of the shading, once per pixel
  {
    float xw[3];
    backproject(q.depth, px, py, cam, xw);
    shade_view(q, xw, cam, sv);
  }
  float sum[3] = {0.f, 0.f, 0.f};  // SSSGS_SUM_LIGHTS: this lane's share of the sum over the lights
#pragma unroll
  for (int l = 0; l < LB; ++l) {
    if (l >= n_lights) break;
    const int64_t fp = (int64_t)l * frame_stride_px + pidx;
    if (gbuf_out) {
      float4* gp = reinterpret_cast<float4*>(gbuf_out + fp * SSSGS_GBUF_CHANNELS);
      if (0 % E == slot) gp[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
      if (1 % E == slot) gp[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
      if (2 % E == slot) gp[2] = make_float4(acc[8], acc[9], accl[l][0], accl[l][1]);
      if (3 % E == slot) gp[3] = make_float4(accl[l][2], accl[l][3], A, T);
    }
    if (l % E != slot) continue;
    float rgb[3], dif[3] = {0.f, 0.f, 0.f}, spc[3] = {0.f, 0.f, 0.f};
    if (covered) {
      const float lsss[3] = {accl[l][0] * iA, accl[l][1] * iA, accl[l][2] * iA};
      shade_light(sv, lsss, accl[l][3] * iA, A, cam, lights.l[l], rgb, dif, spc, sum_mode == 0);
    } else {
      rgb[0] = cam.bg[0]; rgb[1] = cam.bg[1]; rgb[2] = cam.bg[2];
    }
    if (sum_mode != 0) {
      if (covered) { sum[0] += rgb[0]; sum[1] += rgb[1]; sum[2] += rgb[2]; }
      continue;
    }
    if (rgb_out) {
      float* o = rgb_out + fp * 3;
      o[0] = rgb[0]; o[1] = rgb[1]; o[2] = rgb[2];
    }
    if (aovd_out) {
      float* o = aovd_out + fp * 3;
      o[0] = dif[0]; o[1] = dif[1]; o[2] = dif[2];
    }
    if (aovs_out) {
      float* o = aovs_out + fp * 3;
      o[0] = spc[0]; o[1] = spc[1]; o[2] = spc[2];
    }
  }
  if (sum_mode != 0) {
    // the lights were dealt to the E lanes of a pixel: add the shares (all lanes of the warp are
    // still here: `inside` lanes only diverge below), then one lane per pixel writes
    if (E > 1) {
#pragma unroll
      for (int o = P; o < 32; o <<= 1)
#pragma unroll
        for (int c = 0; c < 3; ++c) sum[c] += __shfl_xor_sync(__activemask(), sum[c], o);
    }
    if (slot == 0 && rgb_out) {
      float* o = rgb_out + pidx * 3;
      const float bgw = covered ? 1.f - A : 1.f;  // background term, once per pixel
#pragma unroll
      for (int c = 0; c < 3; ++c) o[c] = sum_mode == 1 ? sum[c] + bgw * cam.bg[c] : o[c] + sum[c];
    }
  }
}

// MARK = true is the visibility pre-pass of a light sweep: the same walk (same culling, alphas,
// transmittance chain and stop rule, hence the same set of blended entries) without channels,
// shading or outputs; it sets contrib[g] = 1 for every Gaussian that is blended at some pixel.  The
// MLP of the sweep then only evaluates those Gaussians (the others are never read by a blend).
// FWD = true is the "w/o deferred" variant (Tab. 2, Fig. 5): Eq. 7 was evaluated
// per Gaussian (shade_gaussians_kernel), the walk composites those RGB values per light (Eq. 3)
// and the epilogue only adds the background: no G-buffer channels, no per-pixel shading.
// `block` = position in the work order (tile_order index * CTAs per tile + sub-region)
template <int LB, int E, int WARPS, int U, bool MARK, bool FWD = false>
__device__ __forceinline__ void
raster_body(const CamParams& cam, const LightBatch& lights, int n_lights,
            const uint2* __restrict__ ranges, const uint32_t* __restrict__ tile_order,
            const uint32_t* __restrict__ sorted_vals,
            const float4* __restrict__ rec_a, const float4* __restrict__ rec_b,
            const float4* __restrict__ attr, const float4* __restrict__ mlp_out,
            float* __restrict__ rgb_out, float* __restrict__ gbuf_out,
            float* __restrict__ aovd_out, float* __restrict__ aovs_out,
            int64_t frame_stride_px, uint8_t* __restrict__ contrib, int sum_mode,
            const WeightCache& wc, const uint32_t* __restrict__ only_if_set, int block) {
  using S = RasterShape<E, WARPS>;
  constexpr int P = S::P, THREADS = S::THREADS;
  constexpr int NC = MARK ? 2 : (FWD ? 2 + LB : 5 + LB);  // float4 components per list entry
  constexpr unsigned FULL = 0xFFFFFFFFu;
  constexpr int NS = raster_stages(LB, MARK, FWD);
  extern __shared__ float4 s_dyn[];
  // a ring of NS stages of component-major entry data, the Gaussian ids of the staged entries (MARK),
  // one hit queue per warp, and the ring's mbarriers: full[s] completes when every thread's copies of a
  // batch have landed in stage s, empty[s] when every warp has finished reading it
  float4 (*s_c)[NC][kBatch] = reinterpret_cast<float4 (*)[NC][kBatch]>(s_dyn);
  uint32_t (*s_gid)[kBatch] = reinterpret_cast<uint32_t (*)[kBatch]>(s_dyn + NS * NC * kBatch);
  uint8_t (*s_q)[kBatch] = reinterpret_cast<uint8_t (*)[kBatch]>(s_gid + NS);
  uint64_t* s_full = reinterpret_cast<uint64_t*>(s_q + WARPS);
  uint64_t* s_empty = s_full + NS;
  uint32_t* s_done = reinterpret_cast<uint32_t*>(s_empty + NS);  // warps whose pixels are all finished

  pdl_prologue();
  if (only_if_set && *only_if_set == 0u) return;  // weight-cache fallback walk, not needed
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int slot = lane / P, pix = lane % P;
  const int tile = (int)tile_order[block / S::SUBS];  // longest lists first
  const int sub = block % S::SUBS;
  const int tx = tile % cam.tiles_x, ty = tile / cam.tiles_x;
  constexpr int WPR = S::RW / S::PW;  // warps per region row
  const int bx = tx * kTile + (sub % S::SX) * S::RW + (warp % WPR) * S::PW;
  const int by = ty * kTile + (sub / S::SX) * S::RH + (warp / WPR) * S::PH;
  const int px = bx + pix % S::PW, py = by + pix / S::PW;
  const bool inside = px < cam.width && py < cam.height;
  const float fpx = (float)px, fpy = (float)py;
  // centre and half-size of this warp's pixel block
  constexpr float bhw = 0.5f * (S::PW - 1), bhh = 0.5f * (S::PH - 1);
  const float bcx = (float)bx + bhw, bcy = (float)by + bhh;

  const uint2 range = ranges[tile];
  float T = 1.f, A = 0.f;  // T is identical in the E lanes of a pixel; A is a per-lane partial sum
  // accumulators of the walk, two per register pair: (n.x, n.y) (n.z, rough) (b.r, b.g) (b.b, metal)
  // (sss, A), per light (L_SSS.r, L_SSS.g) (L_SSS.b, L_in); the depth rides alone
  float acc_depth = 0.f;
  f32x2 pacc[5], paccl[LB][2];
#pragma unroll
  for (int c = 0; c < 5; ++c) pacc[c] = make_float2(0.f, 0.f);
#pragma unroll
  for (int l = 0; l < LB; ++l) paccl[l][0] = paccl[l][1] = make_float2(0.f, 0.f);
  bool done = !inside;
  // weight cache (MARK, E == 1, wc.weights != nullptr): this warp's chain
  const bool caching = MARK && E == 1 && wc.weights != nullptr;
  bool wc_off = !caching;
  uint32_t wc_chunk = 0, wc_items = 0;

  const uint32_t n_entries = range.y - range.x;
  const int n_batches = (int)((n_entries + kBatch - 1) / kBatch);
  if (tid == 0) {
    for (int st = 0; st < NS; ++st) {
      mbar_init(s_full + st, THREADS);
      mbar_init(s_empty + st, WARPS);
    }
    *s_done = 0u;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // ---- staging ring ---------------------------------------------------------------------------
  // Batches of 128 list entries travel through a ring of NS shared-memory stages.  Every thread
  // copies the same slice of every batch (entry tid % 128, components tid / 128, + THREADS / 128, ...)
  // with cp.async and arrives on the stage's `full` barrier when its copies have landed; a warp
  // arrives on `empty` when it has finished a stage.  A warp therefore only ever waits for data,
  // or -- NS batches ahead of the slowest warp of the CTA -- for a free stage: warps whose pixel
  // blocks see few entries run ahead instead of idling at a CTA-wide barrier per batch.
  const int my_e = tid & (kBatch - 1);
  int next_fill = 0;                       // next batch this thread has to copy its slice of
  uint32_t next_gid = (uint32_t)my_e < n_entries ? sorted_vals[range.x + my_e] : 0u;
  auto all_done = [&]() { return *reinterpret_cast<volatile uint32_t*>(s_done) >= (uint32_t)WARPS; };
  // copies this thread's slice of batch next_fill if that batch's stage is free (blocking: wait for it);
  // returns false if nothing was issued
  auto fill = [&](bool blocking) -> bool {
    const int g = next_fill;
    if (g >= n_batches) return false;
    const int st = g % NS;
    if (g >= NS) {  // the stage still holds batch g - NS until every warp has released it
      const uint32_t par = (uint32_t)((g / NS - 1) & 1);
      if (!mbar_test(s_empty + st, par)) {
        if (!blocking) return false;
        while (!mbar_try(s_empty + st, par))  // parked between polls: the issue slots go to the working warps
          if (all_done()) return false;
      }
    }
    if ((uint32_t)(g * kBatch + my_e) < n_entries) {
      const uint32_t gid = next_gid;
      for (int comp = tid / kBatch; comp < NC; comp += THREADS / kBatch) {
        const float4* src;
        if (comp == 0) src = rec_a + gid;
        else if (comp == 1) src = rec_b + gid;
        else if (FWD) src = mlp_out + (size_t)gid * n_lights + min(comp - 2, n_lights - 1);
        else if (comp < 5) src = attr + 3 * (size_t)gid + (comp - 2);
        else src = mlp_out + (size_t)gid * n_lights + min(comp - 5, n_lights - 1);
        cp_async16(&s_c[st][comp][my_e], src);
      }
      if (MARK && tid < kBatch) cp_async4(&s_gid[st][my_e], sorted_vals + range.x + (size_t)g * kBatch + my_e);
    }
    mbar_arrive_on_copies(s_full + st);
    ++next_fill;
    const uint32_t nxt = (uint32_t)(next_fill * kBatch + my_e);
    if (nxt < n_entries) next_gid = sorted_vals[range.x + nxt];
    return true;
  };

  bool counted = false;  // this warp has been added to s_done
  for (int b = 0; b < n_batches; ++b) {
    const int st = b % NS;
    const int cnt = (int)min((uint32_t)kBatch, n_entries - (uint32_t)b * kBatch);
    bool alive = true;
    while (next_fill <= b && alive) alive = fill(true);        // my slice of batch b itself
    if (!alive) break;                                         // every warp of the CTA is finished
    while (next_fill < b + NS && fill(false)) {                // and of the batches ahead, as stages free up
    }
    const bool warp_done = __all_sync(FULL, done);
    if (warp_done) {
      if (!counted) {
        counted = true;
        if (lane == 0) atomicAdd(s_done, 1u);
      }
      if (lane == 0) mbar_arrive(s_empty + st);                // releases the stage without reading it
      if (all_done()) break;
      continue;
    }
    mbar_wait(s_full + st, (uint32_t)((b / NS) & 1));          // every thread's copies of batch b have landed

    // ---- cull: lane <-> entry; queue the entries whose alpha >= 1/255 support box overlaps this
    //      warp's pixel block, in list order --------------------------------------------------------
    int nq = 0;
    for (int c0 = 0; c0 < cnt; c0 += 32) {
      bool hit = false;
      if (c0 + lane < cnt) {
        const float4 ra = s_c[st][0][c0 + lane];
        const float2 ext = __half22float2(*reinterpret_cast<const __half2*>(&ra.w));
        // support box [pix - ext, pix + ext] against the block [bcx - bhw, bcx + bhw] (same in y)
        hit = fabsf(ra.x - bcx) <= ext.x + bhw && fabsf(ra.y - bcy) <= ext.y + bhh;
      }
      const unsigned m = __ballot_sync(FULL, hit);
      if (hit) s_q[warp][nq + __popc(m & ((1u << lane) - 1u))] = (uint8_t)(c0 + lane);
      nq += __popc(m);
    }
    __syncwarp();

    // ---- walk the queue, U groups of E entries at a time --------------------------------------------
    for (int q0 = 0; q0 < nq; q0 += E * U) {
      int j[U];
      float alpha[U], zed[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int qi = q0 + u * E + slot;
        const bool live = qi < nq && !done;
        j[u] = s_q[warp][qi < nq ? qi : q0];
        const float4 ra = s_c[st][0][j[u]];
        const float4 rb = s_c[st][1][j[u]];  // conic pre-scaled for exp2 (see project_kernel)
        const float dx = fpx - ra.x, dy = fpy - ra.y;
        // p = log2(e) * (-1/2 d^T Sigma'^-1 d)
        const float p = fmaf(fmaf(rb.y, dy, rb.x * dx), dx, rb.z * dy * dy);
        const float al = fminf(kAlphaMax, rb.w * ex2_approx(p));
        alpha[u] = (live && p <= 0.f && al >= kAlphaMin) ? al : 0.f;
        zed[u] = ra.z;
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        // front-to-back over the E slots of this group: T_{k+1} = T_k (1 - alpha_k), in list order
        if (done) alpha[u] = 0.f;  // a stop in an earlier group of this iteration
        const float om = 1.f - alpha[u];
        float Tk = T, myT = T;
#pragma unroll
        for (int k = 0; k < E; ++k) {
          const float omk = (E == 1) ? om : __shfl_sync(FULL, om, k * P + pix);
          if (k == slot) myT = Tk;
          Tk *= omk;
        }
        float w;
        if (__any_sync(FULL, Tk < kTMin)) {
          // some pixel crosses T_min inside this group: apply the stop rule entry by entry
          // (the entry that would take T below T_min is not blended, nor is anything behind it)
          float Ts = T;
          bool stop = done, mine = false;
#pragma unroll
          for (int k = 0; k < E; ++k) {
            const float omk = (E == 1) ? om : __shfl_sync(FULL, om, k * P + pix);
            if (!stop && omk < 1.f) {
              const float Tn = Ts * omk;
              if (Tn < kTMin) {
                stop = true;
              } else {
                if (k == slot) { myT = Ts; mine = true; }
                Ts = Tn;
              }
            }
          }
          T = Ts;
          done = stop;
          w = mine ? alpha[u] * myT : 0.f;
        } else {
          T = Tk;
          w = alpha[u] * myT;
        }
        if (MARK) {
          if (!wc_off && __any_sync(FULL, w > 0.f)) {
            const uint32_t in_chunk = wc_items % kWcChunk;
            if (in_chunk == 0) {  // the chain needs a new chunk
              uint32_t c = 0;
              if (lane == 0) c = atomicAdd(wc.chunks, 1u);
              c = __shfl_sync(FULL, c, 0);
              if (c >= wc.capacity) {
                if (lane == 0) *wc.overflow = 1u;
                wc_off = true;
              } else {
                if (lane == 0) {
                  if (wc_items == 0) wc.head[tile * 8 + sub * WARPS + warp] = c;
                  else wc.next[wc_chunk] = c;
                }
                wc_chunk = c;
              }
            }
            if (!wc_off) {
              wc.weights[((size_t)wc_chunk * kWcChunk + in_chunk) * 32 + lane] = w;
              if (lane == 0)
                wc.hdr[(size_t)wc_chunk * kWcChunk + in_chunk] = make_uint2(s_gid[st][j[u]], __float_as_uint(zed[u]));
              ++wc_items;
            }
          }
          if (w > 0.f) contrib[s_gid[st][j[u]]] = 1;
        } else if (FWD) {
          if (__any_sync(FULL, w > 0.f)) {
            const int jj = j[u];
            const f32x2 ww = make_float2(w, w);
#pragma unroll
            for (int l = 0; l < LB; ++l) {
              const float4 c = s_c[st][2 + l][jj];  // per-Gaussian shaded RGB for light l (w = 0)
              fma2(paccl[l][0], ww, c.x, c.y);
              fma2(paccl[l][1], ww, c.z, c.w);
            }
            A += w;
          }
        } else if (__any_sync(FULL, w > 0.f)) {
          const int jj = j[u];
          const float4 a0 = s_c[st][2][jj], a1 = s_c[st][3][jj], a2 = s_c[st][4][jj];
          const f32x2 ww = make_float2(w, w);
          acc_depth = fmaf(w, zed[u], acc_depth);
          fma2(pacc[0], ww, a0.x, a0.y);
          fma2(pacc[1], ww, a0.z, a0.w);
          fma2(pacc[2], ww, a1.x, a1.y);
          fma2(pacc[3], ww, a1.z, a1.w);
          fma2(pacc[4], ww, a2.x, a2.y);  // a2 = (sss, 1, 0, 0): the second half is A += w
#pragma unroll
          for (int l = 0; l < LB; ++l) {
            const float4 mo = s_c[st][5 + l][jj];
            fma2(paccl[l][0], ww, mo.x, mo.y);
            fma2(paccl[l][1], ww, mo.z, mo.w);
          }
        }
      }
      if (__all_sync(FULL, done)) break;
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(s_empty + st);
  }
  cp_async_wait_all();
  if (MARK) {
    if (caching) {
      if (lane == 0) wc.count[tile * 8 + sub * WARPS + warp] = wc_items;
      if (inside) wc.T[(int64_t)py * cam.width + px] = T;
    }
    return;
  }

  raster_finish<LB, E, FWD>(acc_depth, pacc, paccl, A, T, inside, px, py, slot, cam, lights, n_lights, rgb_out,
                            gbuf_out, aovd_out, aovs_out, frame_stride_px, sum_mode);
}

// Copies caller-supplied MLP outputs ([n_light][n][4], light stride given) into the internal
// [n][n_lights] float4 layout the rasteriser gathers from.
__global__ void __launch_bounds__(256)
gather_precomputed_kernel(const float4* __restrict__ pre, int64_t n, int n_lights,
                          int64_t light_stride_f4, float4* __restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (i >= n * n_lights) return;
  const int64_t g = i / n_lights;
  const int l = (int)(i % n_lights);
  out[i] = pre[(int64_t)l * light_stride_f4 + g];
}

}  // namespace

int launch_gather_precomputed(const float* pre, int64_t n, int n_lights, int64_t light_stride,
                              float4* out_internal, cudaStream_t s) {
  if (n == 0) return 0;
  const int64_t total = n * n_lights;
  gather_precomputed_kernel<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(
      reinterpret_cast<const float4*>(pre), n, n_lights, light_stride / 4, out_internal);
  return 1;
}

template <int LB, int E, int WARPS, int U, bool MARK, bool FWD = false>
__global__ void __launch_bounds__(WARPS * 32)
raster_shade_kernel(CamParams cam, LightBatch lights, int n_lights,
                    const uint2* __restrict__ ranges, const uint32_t* __restrict__ tile_order,
                    const uint32_t* __restrict__ sorted_vals,
                    const float4* __restrict__ rec_a, const float4* __restrict__ rec_b,
                    const float4* __restrict__ attr, const float4* __restrict__ mlp_out,
                    float* __restrict__ rgb_out, float* __restrict__ gbuf_out,
                    float* __restrict__ aovd_out, float* __restrict__ aovs_out,
                    int64_t frame_stride_px, uint8_t* __restrict__ contrib, int sum_mode,
                    WeightCache wc, const uint32_t* __restrict__ only_if_set) {
  raster_body<LB, E, WARPS, U, MARK, FWD>(cam, lights, n_lights, ranges, tile_order, sorted_vals, rec_a, rec_b, attr,
                                          mlp_out, rgb_out, gbuf_out, aovd_out, aovs_out, frame_stride_px, contrib,
                                          sum_mode, wc, only_if_set, (int)blockIdx.x);
}

// Small images: the few longest tile lists (the first tiles of the work order, at most cap_long)
// decide when the kernel ends if they are walked like the others.  The first cap_long * 4
// CTAs of this kernel walk them with 4 entry slots per warp and 4 CTAs per tile (half the sequential
// length), the other CTAs walk the remaining tiles with 2 slots and 2 CTAs per tile.
template <int LB, int EL>
__global__ void __launch_bounds__(256)
raster_mixed_kernel(CamParams cam, LightBatch lights, int n_lights,
                    const uint2* __restrict__ ranges, const uint32_t* __restrict__ tile_order,
                    const uint32_t* __restrict__ sorted_vals,
                    const float4* __restrict__ rec_a, const float4* __restrict__ rec_b,
                    const float4* __restrict__ attr, const float4* __restrict__ mlp_out,
                    float* __restrict__ rgb_out, float* __restrict__ gbuf_out,
                    float* __restrict__ aovd_out, float* __restrict__ aovs_out,
                    int64_t frame_stride_px, int sum_mode, const uint32_t* __restrict__ only_if_set,
                    const uint32_t* __restrict__ bucket_starts, int long_log2, int cap_long) {
  pdl_prologue();
  // bucket_starts[k] = tiles with at least 2^k entries (they come first in the work order).  The long
  // class is "at least 2^k entries" for the smallest k >= long_log2 that fits the cap_long * EL CTAs
  // reserved for it: a rule on the list length alone, so that which tiles are walked in which shape
  // (hence the order of their partial sums) does not depend on the arbitrary order inside a bucket.
  int k = long_log2;
  while (k < 31 && bucket_starts[k] > (uint32_t)cap_long) ++k;
  const int n_long = (int)bucket_starts[k];
  const WeightCache none{};
  if ((int)blockIdx.x < cap_long * EL) {
    if ((int)blockIdx.x >= n_long * EL) return;
    raster_body<LB, EL, 8, (EL == 8 ? 1 : 2), false, false>(cam, lights, n_lights, ranges, tile_order, sorted_vals, rec_a, rec_b, attr,
                                           mlp_out, rgb_out, gbuf_out, aovd_out, aovs_out, frame_stride_px, nullptr,
                                           sum_mode, none, only_if_set, (int)blockIdx.x);
  } else {
    const int block = (int)blockIdx.x - cap_long * EL;
    if (block < n_long * 2) return;
    raster_body<LB, 2, 8, 2, false, false>(cam, lights, n_lights, ranges, tile_order, sorted_vals, rec_a, rec_b, attr,
                                           mlp_out, rgb_out, gbuf_out, aovd_out, aovs_out, frame_stride_px, nullptr,
                                           sum_mode, none, only_if_set, block);
  }
}

// Launches one rasteriser variant: LB lights per walk, E entry slots per warp, WARPS warps per CTA.
template <int LB, int E, int WARPS, int U, bool MARK = false, bool FWD = false>
static int launch_variant(const CamParams& cam, const LightBatch& lights, int n_lights,
                          const GeomBuffers& gb, const uint32_t* sorted_vals, const float4* attr,
                          const float4* mlp_out, float* rgb, float* gbuf, float* aov_d, float* aov_s,
                          int64_t frame_stride_px, int tiles, cudaStream_t s, uint8_t* contrib = nullptr,
                          int sum_mode = 0, const WeightCache* wc = nullptr, const uint32_t* only_if_set = nullptr) {
  using S = RasterShape<E, WARPS>;
  constexpr int smem = raster_smem(LB, MARK, FWD, WARPS);
  if (ensure_dyn_smem(reinterpret_cast<const void*>(raster_shade_kernel<LB, E, WARPS, U, MARK, FWD>), smem) != cudaSuccess)
    return -1;
  launch_pdl(raster_shade_kernel<LB, E, WARPS, U, MARK, FWD>, dim3(tiles * S::SUBS), dim3(S::THREADS), smem, s, cam,
             lights, n_lights, gb.ranges, gb.tile_order, sorted_vals, gb.rec_a, gb.rec_b, attr, mlp_out, rgb, gbuf,
             aov_d, aov_s, frame_stride_px, contrib, sum_mode, wc ? *wc : WeightCache{}, only_if_set);
  return 1;
}

constexpr int kLongTilesCap = 64;  // tiles the mixed kernel can walk with 4 CTAs each

template <int LB, int EL>
static int launch_mixed_e(const CamParams& cam, const LightBatch& lights, int n_lights, const GeomBuffers& gb,
                          const uint32_t* sorted_vals, const float4* attr, const float4* mlp_out, float* rgb, float* gbuf,
                          float* aov_d, float* aov_s, int64_t frame_stride_px, int tiles, cudaStream_t s, int sum_mode,
                          const uint32_t* only_if_set, int long_log2) {
  constexpr int smem = raster_smem(LB, false, false, 8);
  if (ensure_dyn_smem(reinterpret_cast<const void*>(raster_mixed_kernel<LB, EL>), smem) != cudaSuccess) return -1;
  launch_pdl(raster_mixed_kernel<LB, EL>, dim3(kLongTilesCap * EL + tiles * 2), dim3(256), smem, s, cam, lights, n_lights,
             gb.ranges, gb.tile_order, sorted_vals, gb.rec_a, gb.rec_b, attr, mlp_out, rgb, gbuf, aov_d, aov_s,
             frame_stride_px, sum_mode, only_if_set, (const uint32_t*)(gb.counters + DC_BUCKET_STARTS), long_log2,
             kLongTilesCap);
  return 1;
}
template <int LB>
static int launch_mixed(const CamParams& cam, const LightBatch& lights, int n_lights, const GeomBuffers& gb,
                        const uint32_t* sorted_vals, const float4* attr, const float4* mlp_out, float* rgb, float* gbuf,
                        float* aov_d, float* aov_s, int64_t frame_stride_px, int tiles, cudaStream_t s, int sum_mode,
                        const uint32_t* only_if_set) {
  static int log2len = -1, el = 4;
  if (log2len < 0) {  // tuning aids
    const char* e = getenv("SSSGS_LONG_LOG2");
    log2len = e ? atoi(e) : kLongListLog2;
    const char* f = getenv("SSSGS_LONG_E");
    el = f ? atoi(f) : 4;
  }
  if (el == 8)
    return launch_mixed_e<LB, 8>(cam, lights, n_lights, gb, sorted_vals, attr, mlp_out, rgb, gbuf, aov_d, aov_s,
                                 frame_stride_px, tiles, s, sum_mode, only_if_set, log2len);
  return launch_mixed_e<LB, 4>(cam, lights, n_lights, gb, sorted_vals, attr, mlp_out, rgb, gbuf, aov_d, aov_s,
                               frame_stride_px, tiles, s, sum_mode, only_if_set, log2len);
}

// Tuning aid: SSSGS_RASTER_MODE = "<E><W>" digits, e.g. "18" (E=1, 8 warps: one CTA per tile, one
// thread per pixel), "48" (E=4, 8 warps: four 8x8-pixel CTAs per tile), "416" (E=4, 16 warps).
static int raster_mode() {
  static int mode = -1;
  if (mode < 0) {
    const char* e = getenv("SSSGS_RASTER_MODE");
    mode = e ? atoi(e) : 0;
  }
  return mode;
}

int launch_raster(const CamParams& cam, const LightBatch& lights, int n_lights,
                  const GeomBuffers& gb, const uint32_t* sorted_vals, const float4* attr,
                  const float4* mlp_out, float* rgb, float* gbuf, float* aov_d, float* aov_s,
                  int64_t frame_stride_px, int sum_mode, cudaStream_t s, const uint32_t* only_if_set) {
  const int tiles = cam.tiles_x * cam.tiles_y;
  if (tiles == 0) return 0;
  // Default shape: few tiles (small images) leave SMs idle behind the longest tile lists, so the
  // lists are walked by 2 CTAs per tile with 2 entry slots per warp (4x4-pixel blocks); with many
  // tiles the classic one-thread-per-pixel shape executes fewer instructions per blended pair
  // (measured: DESIGN.md).
  int mode = raster_mode();
  if (mode == 0) {
    if (tiles <= 1600) {  // 2 slots / 2 CTAs per tile, the longest lists with 4 / 4
      if (n_lights <= 1) return launch_mixed<1>(cam, lights, n_lights, gb, sorted_vals, attr, mlp_out, rgb, gbuf, aov_d, aov_s, frame_stride_px, tiles, s, sum_mode, only_if_set);
      if (n_lights <= 4) return launch_mixed<4>(cam, lights, n_lights, gb, sorted_vals, attr, mlp_out, rgb, gbuf, aov_d, aov_s, frame_stride_px, tiles, s, sum_mode, only_if_set);
      return launch_mixed<8>(cam, lights, n_lights, gb, sorted_vals, attr, mlp_out, rgb, gbuf, aov_d, aov_s, frame_stride_px, tiles, s, sum_mode, only_if_set);
    }
    mode = 18;
  }
#define SSSGS_ARGS cam, lights, n_lights, gb, sorted_vals, attr, mlp_out, rgb, gbuf, aov_d, aov_s, frame_stride_px, tiles, s, nullptr, sum_mode, nullptr, only_if_set
#define SSSGS_BY_LB(E, W, U)                                                   \
  do {                                                                         \
    if (n_lights <= 1) return launch_variant<1, E, W, U>(SSSGS_ARGS);          \
    if (n_lights <= 4) return launch_variant<4, E, W, U>(SSSGS_ARGS);          \
    return launch_variant<8, E, W, U>(SSSGS_ARGS);                             \
  } while (0)
  switch (mode) {
    case 18: SSSGS_BY_LB(1, 8, 4);
    case 28: SSSGS_BY_LB(2, 8, 2);
    case 216: SSSGS_BY_LB(2, 16, 2);
    case 48: SSSGS_BY_LB(4, 8, 2);
    case 416: SSSGS_BY_LB(4, 16, 2);
    case 88: SSSGS_BY_LB(8, 8, 1);
    default: SSSGS_BY_LB(4, 8, 2);
  }
#undef SSSGS_BY_LB
#undef SSSGS_ARGS
}

int raster_reads_unblended_rows(int tiles);

namespace {
// "w/o deferred" variant, step 1: Eq. 7 per Gaussian, at the Gaussian's centre with the Gaussian's
// own normal and material (Tab. 2: shading before rasterisation).  Replaces the MLP
// outputs (L_SSS rgb, L_in) of row (g, l) in place by (intensity * L_out rgb, 0).
__global__ void __launch_bounds__(256)
shade_gaussians_kernel(int64_t n, int n_lights, const float* __restrict__ means,
                       const float4* __restrict__ attr, CamParams cam, LightBatch lights,
                       float4* __restrict__ io) {
  pdl_prologue();
  const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (i >= n * n_lights) return;
  const int64_t g = i / n_lights;
  const int l = (int)(i % n_lights);
  const float4 a0 = attr[3 * g], a1 = attr[3 * g + 1], a2 = attr[3 * g + 2];
  ShadeIn q;
  q.depth = 0.f;
  q.nx = a0.x; q.ny = a0.y; q.nz = a0.z; q.rough = a0.w;
  q.br = a1.x; q.bg = a1.y; q.bb = a1.z; q.metal = a1.w;
  q.sss = a2.x;
  const float4 mo = io[i];
  const float lsss[3] = {mo.x, mo.y, mo.z};
  const float xw[3] = {means[3 * g], means[3 * g + 1], means[3 * g + 2]};
  float rgb[3], dif[3], spc[3];
  shade_point(q, lsss, mo.w, 1.f, xw, cam, lights.l[l], rgb, dif, spc, false);
  io[i] = make_float4(rgb[0], rgb[1], rgb[2], 0.f);
}
}  // namespace

int launch_shade_gaussians(int64_t n, int n_lights, const float* means, const float4* attr,
                           const CamParams& cam, const LightBatch& lights, float4* io, cudaStream_t s) {
  if (n == 0 || n_lights == 0) return 0;
  const int64_t total = n * n_lights;
  launch_pdl(shade_gaussians_kernel, dim3((unsigned)((total + 255) / 256)), dim3(256), 0, s, n, n_lights, means,
             attr, cam, lights, io);
  return 1;
}

// "w/o deferred" variant, step 2: composite the per-Gaussian RGB of every light of the batch.
int launch_raster_forward(const CamParams& cam, int n_lights, const GeomBuffers& gb,
                          const uint32_t* sorted_vals, const float4* shaded, float* rgb,
                          int64_t frame_stride_px, cudaStream_t s) {
  const int tiles = cam.tiles_x * cam.tiles_y;
  if (tiles == 0) return 0;
  LightBatch none;
  memset(&none, 0, sizeof none);
  const bool e1 = !raster_reads_unblended_rows(tiles);
#define SSSGS_FWD(LB)                                                                                     \
  return e1 ? launch_variant<LB, 1, 8, 4, false, true>(cam, none, n_lights, gb, sorted_vals, nullptr, shaded, rgb, \
                                                       nullptr, nullptr, nullptr, frame_stride_px, tiles, s)      \
            : launch_variant<LB, 4, 8, 2, false, true>(cam, none, n_lights, gb, sorted_vals, nullptr, shaded, rgb, \
                                                       nullptr, nullptr, nullptr, frame_stride_px, tiles, s)
  if (n_lights <= 1) SSSGS_FWD(1);
  if (n_lights <= 4) SSSGS_FWD(4);
  SSSGS_FWD(8);
#undef SSSGS_FWD
}

namespace {
// staging buffer of one warp and one 16-entry step of the cached walk: rows [16][4 * RPG] float4 + weights
// (rows per entry: 3 attribute rows + LB MLP rows + the depth row; the MLP rows only in a REST walk)
__host__ __device__ constexpr int cached_rows(int lb, bool rest) { return rest ? lb : lb + 4; }
__host__ __device__ constexpr int cached_buf_bytes(int lb, bool rest) {
  return (kWcChunk / 2) * (4 * ((cached_rows(lb, rest) + 3) / 4)) * 16 + (kWcChunk / 2) * 32 * 4;
}
// Per-light walk of a sweep over the weight cache: one warp per 8x4-pixel block streams the block's
// chain -- per entry (Gaussian id, depth) and the 32 weights -- and blends the entry's channels,
// fetched with warp-uniform loads (a Gaussian's rows are shared by neighbouring blocks and tiles: L1 /
// L2 hits).  Same accumulation order and arithmetic as the list walk: bit-identical frames.
// The sums of the light-independent channels (depth, normal, base colour, roughness, metalness, sss, A)
// are the same for every light batch of the view: the first batch's walk (REST = false) blends all
// channels and stores those sums per pixel (wc.gsum), the later ones (REST = true) blend the MLP
// channels only and read them back.
template <int LB, bool REST>
__global__ void __launch_bounds__(256, 2)
raster_cached_kernel(CamParams cam, LightBatch lights, int n_lights, const uint32_t* __restrict__ tile_order,
                     WeightCache wc, const float4* __restrict__ attr, const float4* __restrict__ mlp_out,
                     float* __restrict__ rgb_out, float* __restrict__ gbuf_out, float* __restrict__ aovd_out,
                     float* __restrict__ aovs_out, int64_t frame_stride_px, int sum_mode) {
  pdl_prologue();
  if (*wc.overflow != 0u) return;  // the pool ran out: the list walk launched next does the work
  using S = RasterShape<1, 8>;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tile = (int)tile_order[blockIdx.x];
  const int tx = tile % cam.tiles_x, ty = tile / cam.tiles_x;
  constexpr int WPR = S::RW / S::PW;
  const int px = tx * kTile + (warp % WPR) * S::PW + lane % S::PW;
  const int py = ty * kTile + (warp / WPR) * S::PH + lane / S::PW;
  const bool inside = px < cam.width && py < cam.height;

  // Blend layout: an entry is 4 * RPG float4 "rows" of channels (3 attribute rows, LB MLP rows, one row
  // holding the depth, padding) and 32 weights.  A lane owns 4 pixels x RPG rows (lane = pixel group * 4
  // + row group), so an entry costs it 1 + RPG 16-byte shared-memory loads for 8 * RPG packed FMAs --
  // the one-pixel-per-lane layout needs 3 + LB broadcast loads for the same FMAs per lane and is bound
  // by the shared-memory return path.  Every (pixel, channel) sum is still one fma per entry in list
  // order: bit-identical to the list walk.  The sums are transposed to one pixel per lane at the end.
  constexpr int ROWS = cached_rows(LB, REST), A0 = REST ? 0 : 3;  // A0 = first MLP row
  constexpr int RPG = (ROWS + 3) / 4;
  constexpr int NR4 = 4 * RPG;
  constexpr int H = kWcChunk / 2;
  constexpr int kBufBytes = cached_buf_bytes(LB, REST);
  static_assert(kBufBytes == H * NR4 * 16 + H * 32 * 4, "staging buffer size");
  static_assert(32 * (NR4 + 1) * 16 <= 2 * kBufBytes, "transpose fits in the warp's staging buffers");
  const int pg = lane >> 2, cg = lane & 3;
  f32x2 acc[4][2 * RPG];
#pragma unroll
  for (int q = 0; q < 4; ++q)
#pragma unroll
    for (int c = 0; c < 2 * RPG; ++c) acc[q][c] = make_float2(0.f, 0.f);

  // The chain is staged in steps of 16 entries (half a cache chunk), double-buffered in this warp's
  // shared memory with cp.async: the rows of the step's entries are gathered by (entry = lane % 16,
  // every other row by lane / 16), its 2 KB of weights copied 4 x 16 B per lane; step j+1 is in flight
  // while step j is blended.  Headers and chunk links run one and two chunks ahead of the walk.
  extern __shared__ float4 s_dyn[];
  char* s_warp = reinterpret_cast<char*>(s_dyn) + warp * 2 * kBufBytes;

  const uint32_t n_items = wc.count[tile * 8 + warp];
  const uint32_t n_steps = (n_items + H - 1) / H, n_chunks = (n_items + kWcChunk - 1) / kWcChunk;
  uint32_t chunk = n_items ? wc.head[tile * 8 + warp] : 0u;
  uint32_t nxt = n_chunks > 1 ? wc.next[chunk] : 0u;
  uint2 hdr_cur = (uint32_t)lane < n_items ? wc.hdr[(size_t)chunk * kWcChunk + lane] : make_uint2(0u, 0u);
  uint2 hdr_nxt = (uint32_t)(kWcChunk + lane) < n_items ? wc.hdr[(size_t)nxt * kWcChunk + lane] : make_uint2(0u, 0u);
  uint32_t nxt2 = n_chunks > 2 ? wc.next[nxt] : 0u;

  auto stage = [&](uint32_t j, uint2 hdr_of_lane, uint32_t chunk_id) {
    const uint32_t m = min((uint32_t)H, n_items - j * H);
    const uint32_t e = lane & (H - 1), part = lane / H, half = j & 1u;
    const size_t g = __shfl_sync(0xFFFFFFFFu, hdr_of_lane.x, half * H + e);
    const float depth = __uint_as_float(__shfl_sync(0xFFFFFFFFu, hdr_of_lane.y, half * H + e));
    char* buf = s_warp + half * kBufBytes;
    float4* rows = reinterpret_cast<float4*>(buf) + e * NR4;
    if (e < m) {
#pragma unroll
      for (int r = 0; r < A0 + LB; ++r) {
        if ((r & 1) != (int)part) continue;
        const float4* src = r < A0 ? attr + 3 * g + r : mlp_out + g * n_lights + min(r - A0, n_lights - 1);
        cp_async16(rows + r, src);
      }
      if (!REST && part == 0) rows[A0 + LB] = make_float4(depth, 0.f, 0.f, 0.f);
    }
    float4* w4 = reinterpret_cast<float4*>(buf + H * NR4 * 16);
    const float4* wsrc = reinterpret_cast<const float4*>(wc.weights + ((size_t)chunk_id * kWcChunk + half * H) * 32);
#pragma unroll
    for (int q = 0; q < 4; ++q)
      if ((uint32_t)(q * 4 + lane / 8) < m) cp_async16(&w4[q * 32 + lane], wsrc + q * 32 + lane);
    asm volatile("cp.async.commit_group;" ::: "memory");
  };

  if (n_steps) stage(0, hdr_cur, chunk);
  for (uint32_t j = 0; j < n_steps; ++j) {
    const uint32_t half = j & 1u;
    if (j + 1 < n_steps) {
      if (half) stage(j + 1, hdr_nxt, nxt);
      else stage(j + 1, hdr_cur, chunk);
      asm volatile("cp.async.wait_group 1;" ::: "memory");
    } else {
      asm volatile("cp.async.wait_group 0;" ::: "memory");
    }
    __syncwarp();  // the step's copies of all lanes have landed
    const uint32_t m = min((uint32_t)H, n_items - j * H);
    const char* buf = s_warp + half * kBufBytes;
    const float4* s_rows = reinterpret_cast<const float4*>(buf) + cg * RPG;       // [entry][NR4]
    const float4* s_w4 = reinterpret_cast<const float4*>(buf + H * NR4 * 16) + pg;  // [entry][8]
#pragma unroll 4
    for (uint32_t k = 0; k < m; ++k) {
      const float4 wv = s_w4[k * 8];
      const float w[4] = {wv.x, wv.y, wv.z, wv.w};
      float4 c[RPG];
#pragma unroll
      for (int r = 0; r < RPG; ++r) c[r] = s_rows[k * NR4 + r];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const f32x2 ww = make_float2(w[q], w[q]);
#pragma unroll
        for (int r = 0; r < RPG; ++r) {
          fma2(acc[q][2 * r], ww, c[r].x, c[r].y);
          fma2(acc[q][2 * r + 1], ww, c[r].z, c[r].w);
        }
      }
    }
    __syncwarp();  // every lane has left this buffer before step j+2 is copied into it
    if (half) {
      const uint32_t ci = j / 2 + 1;  // index of the chunk the walk enters now
      chunk = nxt; hdr_cur = hdr_nxt; nxt = nxt2;
      hdr_nxt = (ci + 1) * kWcChunk + lane < n_items ? wc.hdr[(size_t)nxt * kWcChunk + lane] : make_uint2(0u, 0u);
      nxt2 = ci + 2 < n_chunks ? wc.next[nxt] : 0u;
    }
  }

  // transpose: (4 pixels x RPG rows) per lane -> all rows of one pixel per lane
  float acc_depth;
  f32x2 pacc[5], paccl[LB][2];
  {
    float4* t4 = reinterpret_cast<float4*>(s_warp);
    constexpr int TS = NR4 + 1;  // padded pixel stride: conflict-free 16-byte reads
#pragma unroll
    for (int q = 0; q < 4; ++q)
#pragma unroll
      for (int r = 0; r < RPG; ++r)
        t4[(4 * pg + q) * TS + cg * RPG + r] =
            make_float4(acc[q][2 * r].x, acc[q][2 * r].y, acc[q][2 * r + 1].x, acc[q][2 * r + 1].y);
    __syncwarp();
    const float4* mine = t4 + lane * TS;
    float4 a0, a1, a2;
    float4* gs = wc.gsum + 3 * ((int64_t)min(py, cam.height - 1) * cam.width + min(px, cam.width - 1));
    if (REST) {
      a0 = gs[0]; a1 = gs[1]; a2 = gs[2];
    } else {
      a0 = mine[0]; a1 = mine[1]; a2 = mine[2];
      a2.z = mine[A0 + LB].x;  // the depth sum rides in the free slot of the third row
      if (inside) { gs[0] = a0; gs[1] = a1; gs[2] = a2; }
    }
    pacc[0] = make_float2(a0.x, a0.y); pacc[1] = make_float2(a0.z, a0.w);
    pacc[2] = make_float2(a1.x, a1.y); pacc[3] = make_float2(a1.z, a1.w);
    pacc[4] = make_float2(a2.x, a2.y);
    acc_depth = a2.z;
#pragma unroll
    for (int l = 0; l < LB; ++l) {
      const float4 mo = mine[A0 + l];
      paccl[l][0] = make_float2(mo.x, mo.y);
      paccl[l][1] = make_float2(mo.z, mo.w);
    }
  }
  const float T = inside ? wc.T[(int64_t)py * cam.width + px] : 1.f;
  raster_finish<LB, 1, false>(acc_depth, pacc, paccl, 0.f, T, inside, px, py, 0, cam, lights, n_lights, rgb_out,
                              gbuf_out, aovd_out, aovs_out, frame_stride_px, sum_mode);
}
}  // namespace

int launch_raster_cached(const CamParams& cam, const LightBatch& lights, int n_lights,
                         const GeomBuffers& gb, const WeightCache& wc, const float4* attr,
                         const float4* mlp_out, float* rgb, float* gbuf, float* aov_d, float* aov_s,
                         int64_t frame_stride_px, int sum_mode, int first_batch, cudaStream_t s) {
  const int tiles = cam.tiles_x * cam.tiles_y;
  if (tiles == 0) return 0;
#define SSSGS_CACHED(LB, REST)                                                                              \
  do {                                                                                                      \
    constexpr int smem = 8 * 2 * cached_buf_bytes(LB, REST);                                                \
    if (ensure_dyn_smem(reinterpret_cast<const void*>(raster_cached_kernel<LB, REST>), smem) != cudaSuccess) \
      return -1;                                                                                            \
    launch_pdl(raster_cached_kernel<LB, REST>, dim3(tiles), dim3(256), smem, s, cam, lights, n_lights,      \
               gb.tile_order, wc, attr, mlp_out, rgb, gbuf, aov_d, aov_s, frame_stride_px, sum_mode);       \
  } while (0)
#define SSSGS_CACHED_LB(REST)            \
  do {                                   \
    if (n_lights <= 1) SSSGS_CACHED(1, REST);      \
    else if (n_lights <= 4) SSSGS_CACHED(4, REST); \
    else SSSGS_CACHED(8, REST);          \
  } while (0)
  if (first_batch) SSSGS_CACHED_LB(false);
  else SSSGS_CACHED_LB(true);
#undef SSSGS_CACHED_LB
#undef SSSGS_CACHED
  return 1;
}

// Visibility pre-pass of a light sweep (see raster_shade_kernel, MARK): same tile order and shape
// choice as the render walks.
int launch_mark_contrib(const CamParams& cam, const GeomBuffers& gb, const uint32_t* sorted_vals,
                        uint8_t* contrib, const WeightCache* wc, cudaStream_t s) {
  const int tiles = cam.tiles_x * cam.tiles_y;
  if (tiles == 0) return 0;
  LightBatch none;
  memset(&none, 0, sizeof none);
  int mode = raster_mode();
  if (mode == 0) mode = tiles <= 1600 ? 28 : 18;
  const int e = mode / (mode >= 100 ? 100 : 10);
  static int half_tiles = -1;  // tuning aid: SSSGS_MARK_HALF=0 walks a tile with one 8-warp CTA
  if (half_tiles < 0) { const char* h = getenv("SSSGS_MARK_HALF"); half_tiles = h ? atoi(h) : 1; }
  // the weight cache is organised by the 8x4-pixel blocks of the one-slot shape; two 4-warp CTAs per
  // tile (block = sub * 4 + warp) balance the kernel's tail better than one 8-warp CTA
  if (wc && half_tiles)
    return launch_variant<1, 1, 4, 4, true>(cam, none, 0, gb, sorted_vals, nullptr, nullptr, nullptr, nullptr, nullptr,
                                            nullptr, 0, tiles, s, contrib, 0, wc);
  if (e == 1 || wc)
    return launch_variant<1, 1, 8, 4, true>(cam, none, 0, gb, sorted_vals, nullptr, nullptr, nullptr, nullptr, nullptr,
                                            nullptr, 0, tiles, s, contrib, 0, wc);
  return launch_variant<1, 4, 8, 2, true>(cam, none, 0, gb, sorted_vals, nullptr, nullptr, nullptr, nullptr, nullptr,
                                          nullptr, 0, tiles, s, contrib);
}

// 1 when the render walks of an image of `tiles` tiles use more than one entry slot per warp: a
// blend then also multiplies (by a zero weight) the MLP outputs of entries that contribute nowhere,
// so those rows must hold finite values (the compaction kernel zero-fills them).
int raster_reads_unblended_rows(int tiles) {
  int mode = raster_mode();
  if (mode == 0) mode = tiles <= 1600 ? 28 : 18;
  return mode / (mode >= 100 ? 100 : 10) != 1;
}

}  // namespace sssgs

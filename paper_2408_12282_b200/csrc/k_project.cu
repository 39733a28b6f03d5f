// Projection / culling kernel (hot-path step a3) and the per-Gaussian attribute packer.
//
// EWA projection Sigma' = J W Sigma W^T J^T (Eq. 2), Sigma from scale and unit
// quaternion (L72).  Sort keys and tile rectangles depend on this arithmetic and must be
// bit-exact against the CPU oracle, so the kernel implements the canonical fp32 sequence
// P1..P10 of DESIGN.md with explicit round-to-nearest intrinsics (__fmul_rn, __fadd_rn,
// __fmaf_rn, __fdiv_rn, __fsqrt_rn), which nvcc never contracts or re-associates.
//
// One thread per Gaussian: 44 B read (mean 12, scale 12, quaternion 16, opacity 4),
// 44 B written (2 x float4 record, packed rect, tiles_touched) + 4 B depth key.
// The block also accumulates the four 8-bit digit histograms of the depth keys (used by the
// one-sweep radix sort) with warp-aggregated shared-memory atomics.
#include <cuda_fp16.h>

#include "internal.cuh"

namespace sssgs {

namespace {

__device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ float dot3(const float* a, const float* b) {
  return fma_(a[0], b[0], fma_(a[1], b[1], mul(a[2], b[2])));
}
__device__ __forceinline__ float dot3p(const float* a, const float* b, float c) {
  return fma_(a[0], b[0], fma_(a[1], b[1], fma_(a[2], b[2], c)));
}
__device__ __forceinline__ int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

constexpr int kProjThreads = 256;

__global__ void __launch_bounds__(kProjThreads)
project_kernel(int64_t n, const float* __restrict__ means, const float* __restrict__ scales,
               const float* __restrict__ rotations, const float* __restrict__ opacities,
               CamParams cam, float4* __restrict__ rec_a, float4* __restrict__ rec_b,
               uint2* __restrict__ rect_out, uint32_t* __restrict__ touched_out,
               uint32_t* __restrict__ dkeys, uint32_t* __restrict__ hist,
               uint32_t* __restrict__ counters, int tight) {
  __shared__ uint32_t s_hist[4 * 256];
  pdl_prologue();
  for (int i = threadIdx.x; i < 4 * 256; i += kProjThreads) s_hist[i] = 0;
  __syncthreads();

  // grid-stride over blocks of 256 Gaussians: the block's digit histograms are flushed once
  for (int64_t base = (int64_t)blockIdx.x * kProjThreads; base < n; base += (int64_t)gridDim.x * kProjThreads) {
  const int64_t i = base + threadIdx.x;
  const bool in_range = i < n;
  bool vis = false;
  uint32_t key = 0xFFFFFFFFu;
  float4 ra = make_float4(0.f, 0.f, 0.f, 0.f), rb = make_float4(0.f, 0.f, 0.f, 0.f);
  uint2 rc = make_uint2(0u, 0u);
  uint32_t cnt = 0;

  if (in_range) {
    const float mu[3] = {means[3 * i], means[3 * i + 1], means[3 * i + 2]};
    const float* R = cam.R;
    // P1
    float p[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) p[k] = dot3p(R + 3 * k, mu, cam.t[k]);
    const float z = p[2];
    if (z > cam.znear) {
      // P2
      const float u = __fdiv_rn(p[0], z), w = __fdiv_rn(p[1], z);
      const float pix_x = fma_(cam.fx, u, cam.cx), pix_y = fma_(cam.fy, w, cam.cy);
      // P3
      const float lim_x = mul(kFrustumClamp, cam.tanx), lim_y = mul(kFrustumClamp, cam.tany);
      const float u_cl = fminf(lim_x, fmaxf(-lim_x, u)), w_cl = fminf(lim_y, fmaxf(-lim_y, w));
      const float x_cl = mul(u_cl, z), y_cl = mul(w_cl, z);
      // P4
      const float zz = mul(z, z);
      const float j00 = __fdiv_rn(cam.fx, z), j11 = __fdiv_rn(cam.fy, z);
      const float j02 = -__fdiv_rn(mul(cam.fx, x_cl), zz), j12 = -__fdiv_rn(mul(cam.fy, y_cl), zz);
      // P5
      const float4 q = reinterpret_cast<const float4*>(rotations)[i];
      const float qr = q.x, qx = q.y, qy = q.z, qz = q.w;
      const float xx = mul(qx, qx), yy = mul(qy, qy), zz2 = mul(qz, qz), xy = mul(qx, qy),
                  xz = mul(qx, qz), yz = mul(qy, qz), rx = mul(qr, qx), ry = mul(qr, qy),
                  rz = mul(qr, qz);
      float Rq[9];
      Rq[0] = sub(1.f, mul(2.f, add(yy, zz2)));
      Rq[1] = mul(2.f, sub(xy, rz));
      Rq[2] = mul(2.f, add(xz, ry));
      Rq[3] = mul(2.f, add(xy, rz));
      Rq[4] = sub(1.f, mul(2.f, add(xx, zz2)));
      Rq[5] = mul(2.f, sub(yz, rx));
      Rq[6] = mul(2.f, sub(xz, ry));
      Rq[7] = mul(2.f, add(yz, rx));
      Rq[8] = sub(1.f, mul(2.f, add(xx, yy)));
      const float sc[3] = {scales[3 * i], scales[3 * i + 1], scales[3 * i + 2]};
      float M[9];
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) M[3 * a + b] = mul(Rq[3 * a + b], sc[b]);
      float S[9];
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = a; b < 3; ++b) S[3 * a + b] = S[3 * b + a] = dot3(M + 3 * a, M + 3 * b);
      // P6
      float T0[3], T1[3], g0[3], g1[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        T0[k] = fma_(j02, R[6 + k], mul(j00, R[0 + k]));
        T1[k] = fma_(j12, R[6 + k], mul(j11, R[3 + k]));
      }
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        g0[k] = dot3(S + 3 * k, T0);
        g1[k] = dot3(S + 3 * k, T1);
      }
      const float a = add(dot3(T0, g0), kLowPass);
      const float b = dot3(T1, g0);
      const float c = add(dot3(T1, g1), kLowPass);
      // P7
      const float det = fma_(a, c, -mul(b, b));
      if (det > 0.f) {
        const float id = __fdiv_rn(1.f, det);
        const float con_a = mul(c, id), con_b = -mul(b, id), con_c = mul(a, id);
        // P8
        const float mid = mul(0.5f, add(a, c));
        const float disc = fmaxf(kDiscFloor, fma_(mid, mid, -det));
        const float lam = add(mid, __fsqrt_rn(disc));
        const float rad = mul(kRadiusSigma, __fsqrt_rn(lam));
        // P8b
        if ((fabsf(pix_x) <= 1e9f) && (fabsf(pix_y) <= 1e9f) && (rad <= 1e9f)) {
          // P9
          const float tl = (float)kTile;
          const int x0 = clampi((int)floorf(__fdiv_rn(sub(pix_x, rad), tl)), 0, cam.tiles_x);
          const int x1 = clampi((int)floorf(__fdiv_rn(add(pix_x, rad), tl)) + 1, 0, cam.tiles_x);
          const int y0 = clampi((int)floorf(__fdiv_rn(sub(pix_y, rad), tl)), 0, cam.tiles_y);
          const int y1 = clampi((int)floorf(__fdiv_rn(add(pix_y, rad), tl)) + 1, 0, cam.tiles_y);
          const int c2 = (x1 - x0) * (y1 - y0);
          if (c2 > 0) {
            vis = true;
            cnt = (uint32_t)c2;
            key = __float_as_uint(z);  // P10
            // Half-extents of the alpha >= 1/255 support along x and y (bounding box of the ellipse
            // 1/2 d^T Q d <= tau, tau = ln(255 o)): used ONLY by the rasteriser to skip entries per
            // 8x4 pixel block; never by a key or a rect.  Rounded up (slack 0.1 % + 0.01 px, fp16 rp).
            const float o = opacities[i];
            const float tau = logf(255.f * o);
            float ex = 0.f, ey = 0.f;
            if (tau > 0.f) {
              ex = sqrtf(2.f * tau * a) * 1.001f + 0.01f;
              ey = sqrtf(2.f * tau * c) * 1.001f + 0.01f;
            }
            // beyond the fp16 range the round-up conversion yields +inf = "never cull" (a clamp would drop a
            // huge near-plane splat for blocks far from its centre although its tiles are in the lists)
            const __half2 ext = __halves2half2(__float2half_ru(ex), __float2half_ru(ey));
            ra = make_float4(pix_x, pix_y, z, __uint_as_float(*reinterpret_cast<const uint32_t*>(&ext)));
            int tx0 = x0, tx1 = x1, ty0 = y0, ty1 = y1;
            if (tight) {
              // SSSGS_TIGHT_LISTS: keep only the tiles of the canonical rect that hold a pixel
              // inside the support box [pix - e, pix + e] -- the box the rasteriser culls its 8x4-pixel blocks
              // with (same fp16 half-extents), widened by 0.02 px so that a block test can never pass in a
              // tile dropped here: every tile dropped would have been culled in all of its blocks, hence the
              // image is bit-identical.  Tile t holds the pixel centres 16 t .. 16 t + 15.
              if (o < kAlphaMin) {                     // alpha <= o < 1/255 everywhere: never blended
                tx1 = tx0; ty1 = ty0;
              } else {
                const float2 e = __half22float2(ext);  // +inf beyond the fp16 range: the canonical rect stays
                const float lo_x = ceilf((pix_x - e.x - 0.02f - (float)(kTile - 1)) / tl), hi_x = floorf((pix_x + e.x + 0.02f) / tl);
                const float lo_y = ceilf((pix_y - e.y - 0.02f - (float)(kTile - 1)) / tl), hi_y = floorf((pix_y + e.y + 0.02f) / tl);
                tx0 = max(x0, (int)fmaxf(lo_x, 0.f));
                ty0 = max(y0, (int)fmaxf(lo_y, 0.f));
                tx1 = min(x1, (int)fminf(hi_x, 65535.f) + 1);
                ty1 = min(y1, (int)fminf(hi_y, 65535.f) + 1);
                if (tx1 < tx0) tx1 = tx0;
                if (ty1 < ty0) ty1 = ty0;
              }
              cnt = (uint32_t)((tx1 - tx0) * (ty1 - ty0));
            }
            // the rasteriser evaluates alpha = o * 2^(A' dx^2 + B' dx dy + C' dy^2): conic pre-scaled
            // by log2(e) (and the -1/2); not part of any key or rect
            constexpr float kLog2e = 1.4426950408889634f;
            rb = make_float4(-0.5f * kLog2e * con_a, -kLog2e * con_b, -0.5f * kLog2e * con_c, o);
            rc = make_uint2((uint32_t)tx0 | ((uint32_t)tx1 << 16), (uint32_t)ty0 | ((uint32_t)ty1 << 16));
          }
        }
      }
    }
    rec_a[i] = ra;
    rec_b[i] = rb;
    rect_out[i] = rc;
    touched_out[i] = cnt;
    dkeys[i] = key;
  }

  // digit histograms of the depth key (all n keys take part in the sort; culled -> 0xFFFFFFFF)
  const unsigned active = __ballot_sync(0xFFFFFFFFu, in_range);
  if (in_range) {
    const unsigned lane = threadIdx.x & 31;
    // low digits are spread out: plain shared-memory atomics; the high digits (exponent, top of the
    // mantissa) are usually the same in the whole warp: one atomic then (match.any is slow on sm_100)
#pragma unroll
    for (int d = 0; d < 4; ++d) {
      const uint32_t dig = (key >> (8 * d)) & 255u;
      if (d < 2) {
        atomicAdd(&s_hist[d * 256 + dig], 1u);
      } else {
        const int leader = __ffs(active) - 1;
        const uint32_t dig0 = __shfl_sync(active, dig, leader);
        const bool uniform = __all_sync(active, dig == dig0);
        if (uniform) {
          if ((int)lane == leader) atomicAdd(&s_hist[d * 256 + dig], __popc(active));
        } else {
          atomicAdd(&s_hist[d * 256 + dig], 1u);
        }
      }
    }
  }
  const unsigned vmask = __ballot_sync(0xFFFFFFFFu, vis);
  if ((threadIdx.x & 31) == 0 && vmask) atomicAdd(&counters[DC_NVIS], __popc(vmask));
  }
  __syncthreads();
  for (int k = threadIdx.x; k < 4 * 256; k += kProjThreads) {
    const uint32_t v = s_hist[k];
    if (v) atomicAdd(&hist[k], v);
  }
}

// Light- and view-independent channels packed as 3 x float4 per Gaussian so that the
// rasteriser gathers them with 128-bit loads:
//   a0 = (n.x, n.y, n.z, roughness)  a1 = (b.r, b.g, b.b, metallic)  a2 = (sss, 1, 0, 0)
__global__ void __launch_bounds__(256)
pack_attr_kernel(int64_t n, const float* __restrict__ normals, const float* __restrict__ base,
                 const float* __restrict__ rough, const float* __restrict__ metal,
                 const float* __restrict__ sss, float4* __restrict__ attr) {
  pdl_prologue();
  const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (i >= n) return;
  attr[3 * i + 0] = make_float4(normals[3 * i], normals[3 * i + 1], normals[3 * i + 2], rough[i]);
  attr[3 * i + 1] = make_float4(base[3 * i], base[3 * i + 1], base[3 * i + 2], metal[i]);
  attr[3 * i + 2] = make_float4(sss[i], 1.f, 0.f, 0.f);  // the 1 accumulates the coverage A next to sss
}

}  // namespace

int launch_pack_attr(const sssgs_gaussians& g, float4* attr, cudaStream_t s) {
  if (g.n == 0) return 0;
  const unsigned blocks = (unsigned)((g.n + 255) / 256);
  launch_pdl(pack_attr_kernel, dim3(blocks), dim3(256), 0, s, g.n, g.normals, g.base_color, g.roughness,
             g.metallic, g.subsurface, attr);
  return 1;
}

int launch_project(const sssgs_gaussians& g, const CamParams& cam, const GeomBuffers& gb, int tight,
                   cudaStream_t s) {
  if (g.n == 0) return 0;
  unsigned blocks = (unsigned)((g.n + kProjThreads - 1) / kProjThreads);
  if (blocks > 148 * 8) blocks = 148 * 8;
  launch_pdl(project_kernel, dim3(blocks), dim3(kProjThreads), 0, s, g.n, g.means, g.scales, g.rotations,
             g.opacities, cam, gb.rec_a, gb.rec_b, gb.rect, gb.touched, gb.dkeys[0], gb.hist, gb.counters, tight);
  return 1;
}

}  // namespace sssgs

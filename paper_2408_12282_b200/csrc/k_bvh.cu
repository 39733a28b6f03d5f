// Ray-traced per-Gaussian visibility and its SH fit:
// a linear BVH over the alpha >= 1/255 supports of the Gaussians, built on the device, and one
// traversal per (Gaussian, direction) ray that multiplies the transmittances of the Gaussians it
// meets.  See include/sssgs.h (sssgs_bake_visibility) for the definition, DESIGN.md section 7d for
// the reading of the paper.
//
//   bounds  : box of the centres (ordered-integer atomics)
//   morton  : 30-bit Morton code of every centre + the four 8-bit digit histograms the radix
//             passes of k_sort.cu need; the codes are sorted with the depth-sort passes (stable:
//             equal codes stay in index order, so the tree is deterministic)
//   leaves  : per sorted position: centre, opacity, Sigma^-1 (6), cut-off m2 <= 2 ln(255 o), index;
//             box of the support ellipsoid
//   build   : Karras' radix tree over the sorted codes (ties broken by position), one thread per
//             internal node
//   refit   : bottom-up boxes, second arrival at a node computes it
//   trace   : thread = Gaussian (in Morton order: the rays of a warp start next to each other and
//             share a direction, so they visit the same nodes), loop over the directions; the SH
//             sums are accumulated in direction order by the thread itself (no atomics)
#include "internal.cuh"

namespace sssgs {

namespace {

constexpr int kBvhThreads = 256;
constexpr float kBvhAlphaMin = 1.f / 255.f, kBvhAlphaMax = 0.99f, kBvhTMin = 1e-4f;
constexpr float kBvhY00 = 0.2820948f, kBvhY1 = 0.4886025f;
constexpr float kEmptyBox = 1e30f;

// order-preserving map float -> uint32; every finite float maps above 0, so a zeroed word is
// "nothing yet" for atomicMax
__device__ __forceinline__ uint32_t enc_ordered(float x) {
  const uint32_t u = __float_as_uint(x);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float dec_ordered(uint32_t e) {
  return __uint_as_float((e & 0x80000000u) ? (e & 0x7FFFFFFFu) : ~e);
}
__device__ __forceinline__ bool finite3(float x, float y, float z) {
  return isfinite(x) && isfinite(y) && isfinite(z);
}

// bounds[0..2] = max of enc(x), bounds[3..5] = max of enc(-x)
__global__ void __launch_bounds__(kBvhThreads)
bvh_bounds_kernel(int64_t n, const float* __restrict__ means, uint32_t* __restrict__ bounds) {
  pdl_prologue();
  float hi[3] = {-kEmptyBox, -kEmptyBox, -kEmptyBox}, lo[3] = {kEmptyBox, kEmptyBox, kEmptyBox};
  for (int64_t i = (int64_t)blockIdx.x * kBvhThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kBvhThreads) {
    const float x = means[3 * i], y = means[3 * i + 1], z = means[3 * i + 2];
    if (!finite3(x, y, z)) continue;
    hi[0] = fmaxf(hi[0], x); hi[1] = fmaxf(hi[1], y); hi[2] = fmaxf(hi[2], z);
    lo[0] = fminf(lo[0], x); lo[1] = fminf(lo[1], y); lo[2] = fminf(lo[2], z);
  }
#pragma unroll
  for (int a = 0; a < 3; ++a) {
#pragma unroll
    for (int o = 16; o; o >>= 1) {
      hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xFFFFFFFFu, hi[a], o));
      lo[a] = fminf(lo[a], __shfl_xor_sync(0xFFFFFFFFu, lo[a], o));
    }
  }
  if ((threadIdx.x & 31) == 0) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      atomicMax(&bounds[a], enc_ordered(hi[a]));
      atomicMax(&bounds[3 + a], enc_ordered(-lo[a]));
    }
  }
}

__device__ __forceinline__ uint32_t spread10(uint32_t v) {  // 10 bits -> every third bit
  v = (v * 0x00010001u) & 0xFF0000FFu;
  v = (v * 0x00000101u) & 0x0F00F00Fu;
  v = (v * 0x00000011u) & 0xC30C30C3u;
  v = (v * 0x00000005u) & 0x49249249u;
  return v;
}

__global__ void __launch_bounds__(kBvhThreads)
bvh_morton_kernel(int64_t n, const float* __restrict__ means, const uint32_t* __restrict__ bounds,
                  uint32_t* __restrict__ keys, uint32_t* __restrict__ vals, uint32_t* __restrict__ code_of,
                  uint32_t* __restrict__ hist) {
  pdl_prologue();
  __shared__ uint32_t s_hist[4 * 256];
  for (int i = threadIdx.x; i < 4 * 256; i += kBvhThreads) s_hist[i] = 0;
  __syncthreads();
  float lo[3], inv[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const float h = dec_ordered(bounds[a]);
    lo[a] = -dec_ordered(bounds[3 + a]);
    const float ext = h - lo[a];
    inv[a] = ext > 0.f ? 1024.f / ext : 0.f;
  }
  for (int64_t i = (int64_t)blockIdx.x * kBvhThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kBvhThreads) {
    const float p[3] = {means[3 * i], means[3 * i + 1], means[3 * i + 2]};
    uint32_t code = 0x3FFFFFFFu;  // non-finite centres sort last
    if (finite3(p[0], p[1], p[2])) {
      uint32_t q[3];
#pragma unroll
      for (int a = 0; a < 3; ++a) q[a] = (uint32_t)fminf(1023.f, fmaxf(0.f, (p[a] - lo[a]) * inv[a]));
      code = (spread10(q[0]) << 2) | (spread10(q[1]) << 1) | spread10(q[2]);
    }
    keys[i] = code;
    vals[i] = (uint32_t)i;
    code_of[i] = code;
#pragma unroll
    for (int d = 0; d < 4; ++d) atomicAdd(&s_hist[d * 256 + ((code >> (8 * d)) & 255u)], 1u);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 4 * 256; i += kBvhThreads) {
    const uint32_t v = s_hist[i];
    if (v) atomicAdd(&hist[i], v);
  }
}

// Node numbering: internal nodes 0 .. n-2 (root = 0), leaf of sorted position k = n-1+k.
// box_lo[node] = (min xyz, left child as int bits), box_hi[node] = (max xyz, right child).
__global__ void __launch_bounds__(kBvhThreads)
bvh_leaves_kernel(uint32_t n, const uint32_t* __restrict__ depth_hist, const uint32_t* __restrict__ vals0,
                  const uint32_t* __restrict__ vals1, const uint32_t* __restrict__ code_of,
                  const float* __restrict__ means, const float* __restrict__ scales,
                  const float* __restrict__ rotations, const float* __restrict__ opacities,
                  uint32_t* __restrict__ sorted_codes, uint32_t* __restrict__ sorted_gid,
                  float4* __restrict__ leaf, float4* __restrict__ box_lo, float4* __restrict__ box_hi) {
  pdl_prologue();
  const uint32_t* __restrict__ sorted = (depth_passes_run(depth_hist, n, 4, nullptr) & 1) ? vals1 : vals0;
  const uint32_t k = blockIdx.x * kBvhThreads + threadIdx.x;
  if (k >= n) return;
  const uint32_t g = sorted[k];
  sorted_codes[k] = code_of[g];
  sorted_gid[k] = g;
  const float mx = means[3 * g], my = means[3 * g + 1], mz = means[3 * g + 2];
  const float sx = scales[3 * g], sy = scales[3 * g + 1], sz = scales[3 * g + 2];
  const float qr = rotations[4 * g], qx = rotations[4 * g + 1], qy = rotations[4 * g + 2], qz = rotations[4 * g + 3];
  const float o = opacities[g];
  float R[9];
  R[0] = 1.f - 2.f * (qy * qy + qz * qz); R[1] = 2.f * (qx * qy - qr * qz); R[2] = 2.f * (qx * qz + qr * qy);
  R[3] = 2.f * (qx * qy + qr * qz); R[4] = 1.f - 2.f * (qx * qx + qz * qz); R[5] = 2.f * (qy * qz - qr * qx);
  R[6] = 2.f * (qx * qz - qr * qy); R[7] = 2.f * (qy * qz + qr * qx); R[8] = 1.f - 2.f * (qx * qx + qy * qy);
  const float is[3] = {1.f / (sx * sx), 1.f / (sy * sy), 1.f / (sz * sz)}, s2[3] = {sx * sx, sy * sy, sz * sz};
  float Si[6];  // Sigma^-1 = R S^-2 R^T: xx, xy, xz, yy, yz, zz
  {
    int q = 0;
    for (int a = 0; a < 3; ++a)
      for (int b = a; b < 3; ++b)
        Si[q++] = R[3 * a] * R[3 * b] * is[0] + R[3 * a + 1] * R[3 * b + 1] * is[1] + R[3 * a + 2] * R[3 * b + 2] * is[2];
  }
  // alpha >= 1/255  <=>  m2 <= 2 ln(255 o); the support ellipsoid reaches sqrt(cut Sigma_aa) along axis a
  const float cut = 2.f * logf(255.f * o);
  bool ok = finite3(mx, my, mz) && finite3(sx, sy, sz) && sx > 0.f && sy > 0.f && sz > 0.f && cut >= 0.f && isfinite(cut);
#pragma unroll
  for (int q = 0; q < 6; ++q) ok = ok && isfinite(Si[q]);
  float4 lo = make_float4(kEmptyBox, kEmptyBox, kEmptyBox, 0.f), hi = make_float4(-kEmptyBox, -kEmptyBox, -kEmptyBox, 0.f);
  if (ok) {
    float h[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const float var = R[3 * a] * R[3 * a] * s2[0] + R[3 * a + 1] * R[3 * a + 1] * s2[1] + R[3 * a + 2] * R[3 * a + 2] * s2[2];
      h[a] = sqrtf(cut * var) * 1.0001f + 1e-7f * (fabsf(a == 0 ? mx : (a == 1 ? my : mz)) + 1.f);
    }
    lo = make_float4(mx - h[0], my - h[1], mz - h[2], 0.f);
    hi = make_float4(mx + h[0], my + h[1], mz + h[2], 0.f);
  }
  leaf[3 * (size_t)k] = make_float4(mx, my, mz, ok ? o : 0.f);
  leaf[3 * (size_t)k + 1] = make_float4(Si[0], Si[1], Si[2], Si[3]);
  leaf[3 * (size_t)k + 2] = make_float4(Si[4], Si[5], cut, __uint_as_float(g));
  box_lo[n - 1 + k] = lo;
  box_hi[n - 1 + k] = hi;
}

// length of the common prefix of the (code, position) keys of sorted positions i and j; -1 outside
__device__ __forceinline__ int bvh_delta(const uint32_t* __restrict__ codes, int n, int i, int j) {
  if (j < 0 || j >= n) return -1;
  const uint32_t a = codes[i], b = codes[j];
  return a != b ? __clz(a ^ b) : 32 + __clz((uint32_t)i ^ (uint32_t)j);
}

__global__ void __launch_bounds__(kBvhThreads)
bvh_build_kernel(int n, const uint32_t* __restrict__ codes, float4* __restrict__ box_lo,
                 float4* __restrict__ box_hi, int* __restrict__ parent) {
  pdl_prologue();
  const int i = blockIdx.x * kBvhThreads + threadIdx.x;
  if (i >= n - 1) return;
  const int d = bvh_delta(codes, n, i, i + 1) - bvh_delta(codes, n, i, i - 1) >= 0 ? 1 : -1;
  const int dmin = bvh_delta(codes, n, i, i - d);
  int lmax = 2;
  while (bvh_delta(codes, n, i, i + lmax * d) > dmin) lmax *= 2;
  int l = 0;
  for (int t = lmax / 2; t >= 1; t /= 2)
    if (bvh_delta(codes, n, i, i + (l + t) * d) > dmin) l += t;
  const int j = i + l * d;
  const int dnode = bvh_delta(codes, n, i, j);
  int s = 0;
  for (int t = (l + 1) / 2;; t = (t + 1) / 2) {
    if (bvh_delta(codes, n, i, i + (s + t) * d) > dnode) s += t;
    if (t <= 1) break;
  }
  const int gamma = i + s * d + min(d, 0);
  const int left = min(i, j) == gamma ? n - 1 + gamma : gamma;
  const int right = max(i, j) == gamma + 1 ? n - 1 + gamma + 1 : gamma + 1;
  box_lo[i].w = __int_as_float(left);
  box_hi[i].w = __int_as_float(right);
  parent[left] = i;
  parent[right] = i;
  if (i == 0) parent[0] = -1;
}

__global__ void __launch_bounds__(kBvhThreads)
bvh_refit_kernel(int n, float4* box_lo, float4* box_hi, const int* __restrict__ parent, uint32_t* flags) {
  pdl_prologue();
  const int k = blockIdx.x * kBvhThreads + threadIdx.x;
  if (k >= n) return;
  int node = parent[n - 1 + k];
  while (node >= 0) {
    __threadfence();
    if (atomicAdd(&flags[node], 1u) == 0u) return;  // the sibling subtree is not done yet
    __threadfence();
    const int l = __float_as_int(__ldcg(&box_lo[node].w)), r = __float_as_int(__ldcg(&box_hi[node].w));
    const float4 a = __ldcg(&box_lo[l]), b = __ldcg(&box_lo[r]), c = __ldcg(&box_hi[l]), e = __ldcg(&box_hi[r]);
    float4 lo = make_float4(fminf(a.x, b.x), fminf(a.y, b.y), fminf(a.z, b.z), __int_as_float(l));
    float4 hi = make_float4(fmaxf(c.x, e.x), fmaxf(c.y, e.y), fmaxf(c.z, e.z), __int_as_float(r));
    __stcg(&box_lo[node], lo);
    __stcg(&box_hi[node], hi);
    node = parent[node];
  }
}

// slab test of the ray o + t w, t >= 0 (iw = 1 / w, components of w nudged away from 0): entry
// distance, or -1 on a miss
template <bool POS>
__device__ __forceinline__ float hit_box(const float4& lo, const float4& hi, const float o[3], const float iw[3],
                                         float t_max) {
  const float tx0 = (lo.x - o[0]) * iw[0], tx1 = (hi.x - o[0]) * iw[0];
  const float ty0 = (lo.y - o[1]) * iw[1], ty1 = (hi.y - o[1]) * iw[1];
  const float tz0 = (lo.z - o[2]) * iw[2], tz1 = (hi.z - o[2]) * iw[2];
  const float tn = fmaxf(fmaxf(fminf(tx0, tx1), fminf(ty0, ty1)), fmaxf(fminf(tz0, tz1), 0.f));
  float tf = fminf(fminf(fmaxf(tx0, tx1), fmaxf(ty0, ty1)), fmaxf(tz0, tz1));
  if (POS) tf = fminf(tf, t_max);
  // an inverted box is empty (Gaussians that never reach alpha_min)
  return (tn <= tf && lo.x <= hi.x) ? tn : -1.f;
}

constexpr int kBvhStack = 96;

template <bool POS>
__global__ void __launch_bounds__(128)
bvh_trace_kernel(int n, const uint32_t* __restrict__ sorted_gid, const float4* __restrict__ leaf,
                 const float4* __restrict__ box_lo, const float4* __restrict__ box_hi, int n_dirs,
                 const float* __restrict__ dirs, const float* __restrict__ weights, float t_min, int n_coef,
                 float* __restrict__ sh_out, float* __restrict__ vis_out, int dirs_per_group,
                 float4* __restrict__ partial) {
  pdl_prologue();
  const int k = blockIdx.x * 128 + threadIdx.x;
  if (k >= n) return;
  // blockIdx.y = group of directions (more threads for small scenes); a group's sums go to `partial`
  const int dir_begin = blockIdx.y * dirs_per_group, dir_end = min(n_dirs, dir_begin + dirs_per_group);
  const uint32_t gid = sorted_gid[k];
  const float4 me = leaf[3 * (size_t)k];
  float c0 = 0.f, c1 = 0.f, c2 = 0.f, c3 = 0.f;
  int stack[kBvhStack];
  for (int dk = dir_begin; dk < dir_end; ++dk) {
    float w[3] = {dirs[3 * dk], dirs[3 * dk + 1], dirs[3 * dk + 2]};
    float t_max = 3.0e38f;
    if (POS) {  // the ray ends at the point dirs[dk]
      w[0] -= me.x; w[1] -= me.y; w[2] -= me.z;
      const float d = sqrtf(w[0] * w[0] + w[1] * w[1] + w[2] * w[2]);
      const float id = d > 0.f ? 1.f / d : 0.f;
      w[0] *= id; w[1] *= id; w[2] *= id;
      t_max = d - t_min;
    }
    const float o[3] = {fmaf(t_min, w[0], me.x), fmaf(t_min, w[1], me.y), fmaf(t_min, w[2], me.z)};
    float iw[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) iw[a] = 1.f / (fabsf(w[a]) < 1e-20f ? copysignf(1e-20f, w[a]) : w[a]);
    float T = 1.f;
    if (n >= 2 && finite3(o[0], o[1], o[2]) && (!POS || t_max > 0.f)) {
      int sp = 0;
      // nearer child first: the opaque surface next to the ray's start ends most blocked rays early
      // (the product is order independent, the early exit is not a change of the result)
      auto leaf_hit = [&](int c) -> bool {  // true: the ray is extinguished
        const size_t j = (size_t)(c - (n - 1));
        const float4 l0 = leaf[3 * j], l1 = leaf[3 * j + 1], l2 = leaf[3 * j + 2];
        if (__float_as_uint(l2.w) == gid) return false;
        // point of the largest response along the ray, clamped to its start
        const float d[3] = {o[0] - l0.x, o[1] - l0.y, o[2] - l0.z};
        const float Sw[3] = {l1.x * w[0] + l1.y * w[1] + l1.z * w[2], l1.y * w[0] + l1.w * w[1] + l2.x * w[2],
                             l1.z * w[0] + l2.x * w[1] + l2.y * w[2]};
        const float Sd[3] = {l1.x * d[0] + l1.y * d[1] + l1.z * d[2], l1.y * d[0] + l1.w * d[1] + l2.x * d[2],
                             l1.z * d[0] + l2.x * d[1] + l2.y * d[2]};
        const float ww = w[0] * Sw[0] + w[1] * Sw[1] + w[2] * Sw[2];
        const float wd = w[0] * Sd[0] + w[1] * Sd[1] + w[2] * Sd[2];
        const float t = POS ? fminf(t_max, fmaxf(0.f, -wd / ww)) : fmaxf(0.f, -wd / ww);
        const float e[3] = {fmaf(t, w[0], d[0]), fmaf(t, w[1], d[1]), fmaf(t, w[2], d[2])};
        const float m2 = e[0] * (l1.x * e[0] + l1.y * e[1] + l1.z * e[2]) + e[1] * (l1.y * e[0] + l1.w * e[1] + l2.x * e[2]) +
                         e[2] * (l1.z * e[0] + l2.x * e[1] + l2.y * e[2]);
        const float a = l0.w * __expf(-0.5f * m2);
        if (!(a >= kBvhAlphaMin)) return false;
        T *= 1.f - fminf(a, kBvhAlphaMax);
        return T < kBvhTMin;
      };
      int node = 0;
      while (true) {
        const int cl = __float_as_int(box_lo[node].w), cr = __float_as_int(box_hi[node].w);
        float tl = hit_box<POS>(box_lo[cl], box_hi[cl], o, iw, t_max), tr = hit_box<POS>(box_lo[cr], box_hi[cr], o, iw, t_max);
        bool dead = false;
        if (tl >= 0.f && cl >= n - 1) { dead = leaf_hit(cl); tl = -1.f; }
        if (!dead && tr >= 0.f && cr >= n - 1) { dead = leaf_hit(cr); tr = -1.f; }
        if (dead) break;
        if (tl >= 0.f && tr >= 0.f) {
          const bool left_first = tl <= tr;
          if (sp < kBvhStack) stack[sp++] = left_first ? cr : cl;
          node = left_first ? cl : cr;
        } else if (tl >= 0.f) {
          node = cl;
        } else if (tr >= 0.f) {
          node = cr;
        } else {
          if (!sp) break;
          node = stack[--sp];
        }
      }
    }
    const float V = T >= kBvhTMin ? T : 0.f;
    if (vis_out) vis_out[(size_t)gid * n_dirs + dk] = V;
    const float wv = weights[dk] * V;
    c0 = fmaf(wv, kBvhY00, c0);
    c1 = fmaf(wv * kBvhY1, w[1], c1);
    c2 = fmaf(wv * kBvhY1, w[2], c2);
    c3 = fmaf(wv * kBvhY1, w[0], c3);
  }
  if (partial) {
    partial[(size_t)blockIdx.y * n + gid] = make_float4(c0, c1, c2, c3);
  } else if (n_coef == 1) {
    sh_out[gid] = c0;
  } else {
    reinterpret_cast<float4*>(sh_out)[gid] = make_float4(c0, c1, c2, c3);
  }
}

// sums the direction groups' partial SH sums in group order (deterministic)
__global__ void __launch_bounds__(kBvhThreads)
bvh_sh_reduce_kernel(int n, int groups, const float4* __restrict__ partial, int n_coef, float* __restrict__ sh_out) {
  pdl_prologue();
  const int g = blockIdx.x * kBvhThreads + threadIdx.x;
  if (g >= n) return;
  float4 c = partial[g];
  for (int q = 1; q < groups; ++q) {
    const float4 p = partial[(size_t)q * n + g];
    c.x += p.x; c.y += p.y; c.z += p.z; c.w += p.w;
  }
  if (n_coef == 1) sh_out[g] = c.x;
  else reinterpret_cast<float4*>(sh_out)[g] = c;
}

}  // namespace

int launch_bvh_bounds(int64_t n, const float* means, uint32_t* bounds, int max_blocks, cudaStream_t s) {
  int64_t blocks = (n + kBvhThreads - 1) / kBvhThreads;
  if (blocks > max_blocks) blocks = max_blocks;
  launch_pdl(bvh_bounds_kernel, dim3((unsigned)blocks), dim3(kBvhThreads), 0, s, n, means, bounds);
  return 1;
}

int launch_bvh_morton(int64_t n, const float* means, const uint32_t* bounds, uint32_t* keys, uint32_t* vals,
                      uint32_t* code_of, uint32_t* hist, int max_blocks, cudaStream_t s) {
  int64_t blocks = (n + kBvhThreads - 1) / kBvhThreads;
  if (blocks > max_blocks) blocks = max_blocks;
  launch_pdl(bvh_morton_kernel, dim3((unsigned)blocks), dim3(kBvhThreads), 0, s, n, means, bounds, keys, vals, code_of, hist);
  return 1;
}

int launch_bvh_build(const sssgs_gaussians& g, const BvhBuffers& b, const uint32_t* depth_hist,
                     const uint32_t* vals0, const uint32_t* vals1, cudaStream_t s) {
  const uint32_t n = (uint32_t)g.n;
  const unsigned blocks = (n + kBvhThreads - 1) / kBvhThreads;
  launch_pdl(bvh_leaves_kernel, dim3(blocks), dim3(kBvhThreads), 0, s, n, depth_hist, vals0, vals1,
             (const uint32_t*)b.code_of, g.means, g.scales, g.rotations, g.opacities, b.sorted_codes, b.sorted_gid,
             b.leaf, b.box_lo, b.box_hi);
  if (n < 2) return 1;
  launch_pdl(bvh_build_kernel, dim3(blocks), dim3(kBvhThreads), 0, s, (int)n, (const uint32_t*)b.sorted_codes, b.box_lo,
             b.box_hi, b.parent);
  launch_pdl(bvh_refit_kernel, dim3(blocks), dim3(kBvhThreads), 0, s, (int)n, b.box_lo, b.box_hi, (const int*)b.parent,
             b.flags);
  return 3;
}

int launch_bvh_trace(int64_t n, const BvhBuffers& b, int n_dirs, const float* dirs, const float* weights, float t_min,
                     int n_coef, float* sh_out, float* vis_out, int positions, int num_sms, float4* scratch,
                     size_t scratch_bytes, cudaStream_t s) {
  // enough threads to fill the device: split the directions in groups when there are few Gaussians
  int groups = (int)(((int64_t)num_sms * 2048 * 2 + n - 1) / n);
  if (groups > 8) groups = 8;
  if (groups > n_dirs) groups = n_dirs;
  if ((size_t)groups * n * 16 > scratch_bytes) groups = 1;
  const int per = (n_dirs + groups - 1) / groups;
  groups = (n_dirs + per - 1) / per;
  const unsigned blocks = (unsigned)((n + 127) / 128);
  if (positions)
    launch_pdl(bvh_trace_kernel<true>, dim3(blocks, groups), dim3(128), 0, s, (int)n, (const uint32_t*)b.sorted_gid,
               (const float4*)b.leaf, (const float4*)b.box_lo, (const float4*)b.box_hi, n_dirs, dirs, weights, t_min,
               n_coef, sh_out, vis_out, per, groups > 1 ? scratch : (float4*)nullptr);
  else
    launch_pdl(bvh_trace_kernel<false>, dim3(blocks, groups), dim3(128), 0, s, (int)n, (const uint32_t*)b.sorted_gid,
               (const float4*)b.leaf, (const float4*)b.box_lo, (const float4*)b.box_hi, n_dirs, dirs, weights, t_min,
               n_coef, sh_out, vis_out, per, groups > 1 ? scratch : (float4*)nullptr);
  if (groups == 1) return 1;
  launch_pdl(bvh_sh_reduce_kernel, dim3((unsigned)((n + kBvhThreads - 1) / kBvhThreads)), dim3(kBvhThreads), 0, s, (int)n,
             groups, (const float4*)scratch, n_coef, sh_out);
  return 2;
}

}  // namespace sssgs

// Joint SSS / incident-light MLP on the 5th-generation tensor cores (hot-path steps a1 + a2).
//
// (L_SSS, L_in) = f_Theta(mu, Sigma, n, w_in, w_out, v) evaluated per Gaussian for a given view
// and point light (Eq. 6; widths and input list L347).  It is a dense batched
// contraction [rows x K] . [K x N] per layer, so it runs as tcgen05.mma (bf16 x bf16 -> fp32):
//
//   * persistent CTAs, one per SM; ALL layer weights live in shared memory for the whole kernel
//     as UMMA operands (K-major, 128-byte swizzle), packed once per call by mlp_pack_kernel;
//   * a row tile = 128 Gaussians x 1 light = the M of one tcgen05.mma (cta_group::1, M=128);
//     its fp32 accumulator [128 x N] sits in TMEM (one 256-column slot per tile in flight);
//   * two tiles are in flight per CTA ("slots"): while the four epilogue warps of slot 0 read
//     their accumulator back (tcgen05.ld), add the bias, apply the activation, round to bf16 and
//     write the NEXT layer's A operand straight into shared memory in the UMMA swizzled layout,
//     the tensor core runs slot 1's layer -- activations never touch HBM;
//   * the layer-0 A tile is COMPUTED, not loaded: the same warps assemble the 40+F inputs
//     (unit directions, light distance, SH visibility, Fourier encoding of mu) in fp32 and store
//     them as bf16;
//   * warp 8 issues the MMAs (one elected thread) and owns the TMEM allocation; mbarriers
//     (a_ready: 128 arrivals, d_ready: tcgen05.commit) hand tiles back and forth.
//
// Output: float4 (L_SSS rgb, L_in) per (Gaussian, light), 16 B per row.
#include <cuda_bf16.h>

#include "internal.cuh"

namespace sssgs {

namespace {

constexpr int kMlpThreads = 288;       // 2 x 4 epilogue warps + 1 MMA warp
constexpr int kRows = 128;             // rows per tile = UMMA M
constexpr int kSlotCols = 256;         // TMEM columns per slot
constexpr int kKBlockBytes = kRows * 128;  // one 64-wide K block of an A tile (128 rows x 128 B)
constexpr float kY00 = 0.2820948f, kY1 = 0.4886025f;

// ---------------------------------------------------------------------------------------------
// PTX wrappers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(bar)
               : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {
  }
}
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void fence_barrier_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_before() {
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_after() {
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem),
               "r"(ncols)
               : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols)
               : "memory");
}
// D[tmem] (+)= A[smem desc] . B[smem desc]^T, kind::f16 (bf16 inputs, fp32 accumulate)
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b,
                                          uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar)
               : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float* v) {
  uint32_t r[16];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]),
        "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]),
        "=r"(r[14]), "=r"(r[15])
      : "r"(taddr)
      : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}

// UMMA shared-memory descriptor: K-major operand, 128-byte swizzle, rows of 128 B, 8-row groups
// 1024 B apart (SBO), LBO = 1 (unused for swizzled K-major), descriptor version 1 (sm_100).
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr >> 4) & 0x3FFFu);
  d |= (uint64_t)1 << 16;              // leading byte offset (>>4)
  d |= (uint64_t)(1024 >> 4) << 32;    // stride byte offset (>>4)
  d |= (uint64_t)1 << 46;              // version
  d |= (uint64_t)2 << 61;              // SWIZZLE_128B
  return d;
}
// Instruction descriptor: D = F32, A = B = BF16, both K-major, M = 128, N = n.
__device__ __forceinline__ uint32_t make_idesc(int n) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(kRows >> 4) << 24);
}

__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
  __nv_bfloat162 h = __floats2bfloat162_rn(a, b);  // .x = a (low half), .y = b
  return *reinterpret_cast<uint32_t*>(&h);
}
// byte offset of 16-byte chunk `c` (8 bf16 = columns 8c..8c+7) of row `r` inside a K-major
// SWIZZLE_128B operand whose 64-column K blocks are `rows*128` bytes apart
__device__ __forceinline__ uint32_t swz_off(int r, int c, int kblock_bytes) {
  return (uint32_t)((c >> 3) * kblock_bytes + r * 128 + (((c & 7) ^ (r & 7)) << 4));
}

// ---------------------------------------------------------------------------------------------
// Weight packer: caller's W[out][in] (+ bias) -> bf16 UMMA operands in the swizzled layout.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
mlp_pack_kernel(MlpPlan plan, const void* __restrict__ params, int dtype, uint8_t* __restrict__ blob,
                float* __restrict__ bias) {
  auto load = [&](int off) -> float {
    if (dtype == SSSGS_BF16)
      return __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(params)[off]);
    return reinterpret_cast<const float*>(params)[off];
  };
  for (int s = 0; s < plan.n_stages; ++s) {
    const MlpStage st = plan.st[s];
    const int chunks_per_row = ((st.k_pad + 63) / 64) * 8;
    const int total = st.n_pad * chunks_per_row;
    for (int q = blockIdx.x * 256 + threadIdx.x; q < total; q += gridDim.x * 256) {
      const int r = q / chunks_per_row, c = q % chunks_per_row;
      int src = -1;
      if (r < st.src_rows[0]) src = st.src_w[0] + r * st.src_k;
      else if (r < st.src_rows[0] + st.src_rows[1]) src = st.src_w[1] + (r - st.src_rows[0]) * st.src_k;
      float v[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        const int k = c * 8 + e;
        v[e] = (src >= 0 && k < st.src_k) ? load(src + k) : 0.f;
      }
      uint4 pk = make_uint4(pack_bf16(v[0], v[1]), pack_bf16(v[2], v[3]), pack_bf16(v[4], v[5]),
                            pack_bf16(v[6], v[7]));
      *reinterpret_cast<uint4*>(blob + st.w_off + swz_off(r, c, st.n_pad * 128)) = pk;
    }
    for (int r = blockIdx.x * 256 + threadIdx.x; r < st.n_pad; r += gridDim.x * 256) {
      float b = 0.f;
      if (r < st.src_rows[0]) b = load(st.src_b[0] + r);
      else if (r < st.src_rows[0] + st.src_rows[1]) b = load(st.src_b[1] + (r - st.src_rows[0]));
      bias[st.b_off + r] = b;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// The MLP kernel
// ---------------------------------------------------------------------------------------------
struct MlpArgs {
  int64_t n;
  const float *means, *normals, *rotations, *scales, *vis_sh, *feat;
  int sh_coefs;  // 1 (degree 0) or 4 (degree 1)
  float cam_pos[3];
  LightBatch lights;
  int n_lights;
  const uint8_t* blob;
  const float* bias;
  float4* out_internal;        // [n][n_lights]
  float* out_user;             // optional: light l at out_user + l*user_light_stride, [n][4]
  int64_t user_light_stride;   // in floats
  MlpPlan plan;
};

__device__ __forceinline__ float act_fn(float v, int activation, float slope) {
  return v > 0.f ? v : (activation == SSSGS_ACT_LEAKY_RELU ? slope * v : 0.f);
}

// Step a1: assemble the input row of Gaussian g for one light and store it as bf16 into row r
// of the A tile.  Row layout (S1/S13/S14):
//   [ n(3) | rot(2) | scale(3) | w_in(3) | w_out(3) | d | v | gamma(mu)(24) | feat(F) | 0-pad ]
__device__ __forceinline__ void assemble_row(const MlpArgs& a, int64_t g, const LightParams& lt,
                                             uint8_t* A, int r) {
  const float mx = a.means[3 * g], my = a.means[3 * g + 1], mz = a.means[3 * g + 2];
  const float4 q = reinterpret_cast<const float4*>(a.rotations)[g];
  const float sgn = q.x < 0.f ? -1.f : 1.f;
  {
    const uint4 c0 = make_uint4(pack_bf16(a.normals[3 * g], a.normals[3 * g + 1]),
                                pack_bf16(a.normals[3 * g + 2], sgn * q.x),
                                pack_bf16(sgn * q.y, a.scales[3 * g]),
                                pack_bf16(a.scales[3 * g + 1], a.scales[3 * g + 2]));
    *reinterpret_cast<uint4*>(A + swz_off(r, 0, kKBlockBytes)) = c0;
  }
  {
    float wix = lt.pos[0] - mx, wiy = lt.pos[1] - my, wiz = lt.pos[2] - mz;
    const float d = sqrtf(wix * wix + wiy * wiy + wiz * wiz);
    const float id = 1.f / d;
    wix *= id; wiy *= id; wiz *= id;
    float wox = a.cam_pos[0] - mx, woy = a.cam_pos[1] - my, woz = a.cam_pos[2] - mz;
    const float io = 1.f / sqrtf(wox * wox + woy * woy + woz * woz);
    wox *= io; woy *= io; woz *= io;
    float v;
    if (a.sh_coefs == 4) {
      const float4 sh = reinterpret_cast<const float4*>(a.vis_sh)[g];
      v = kY00 * sh.x + kY1 * (sh.y * wiy + sh.z * wiz + sh.w * wix);
    } else {
      v = kY00 * a.vis_sh[g];
    }
    v = fminf(1.f, fmaxf(0.f, v));
    const uint4 c1 = make_uint4(pack_bf16(wix, wiy), pack_bf16(wiz, wox), pack_bf16(woy, woz),
                                pack_bf16(d, v));
    *reinterpret_cast<uint4*>(A + swz_off(r, 1, kKBlockBytes)) = c1;
  }
  {
    // gamma(mu): for k = 0..3: [sin(2^k pi mu_xyz), cos(2^k pi mu_xyz)]; sin(pi x) via sincospif
    float ga[24];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const float f = (float)(1 << k);
      sincospif(f * mx, &ga[6 * k + 0], &ga[6 * k + 3]);
      sincospif(f * my, &ga[6 * k + 1], &ga[6 * k + 4]);
      sincospif(f * mz, &ga[6 * k + 2], &ga[6 * k + 5]);
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const uint4 cc = make_uint4(pack_bf16(ga[8 * c], ga[8 * c + 1]), pack_bf16(ga[8 * c + 2], ga[8 * c + 3]),
                                  pack_bf16(ga[8 * c + 4], ga[8 * c + 5]), pack_bf16(ga[8 * c + 6], ga[8 * c + 7]));
      *reinterpret_cast<uint4*>(A + swz_off(r, 2 + c, kKBlockBytes)) = cc;
    }
  }
  const int F = a.plan.feat_dim;
  const int nchunks = a.plan.in_pad >> 3;
  for (int c = 5; c < nchunks; ++c) {
    const int j = (c - 5) * 8;
    float4 f0 = make_float4(0.f, 0.f, 0.f, 0.f), f1 = f0;
    if (j < F) f0 = *reinterpret_cast<const float4*>(a.feat + g * F + j);
    if (j + 4 < F) f1 = *reinterpret_cast<const float4*>(a.feat + g * F + j + 4);
    const uint4 cc = make_uint4(pack_bf16(f0.x, f0.y), pack_bf16(f0.z, f0.w), pack_bf16(f1.x, f1.y),
                                pack_bf16(f1.z, f1.w));
    *reinterpret_cast<uint4*>(A + swz_off(r, c, kKBlockBytes)) = cc;
  }
}

__global__ void __launch_bounds__(kMlpThreads, 1) mlp_kernel(const __grid_constant__ MlpArgs a) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  const MlpPlan& plan = a.plan;
  const int a_bytes = plan.max_k_bytes;
  uint8_t* sW = smem;
  uint8_t* sA[2] = {smem + plan.blob_bytes, smem + plan.blob_bytes + a_bytes};
  float* sBias = reinterpret_cast<float*>(smem + plan.blob_bytes + 2 * a_bytes);
  uint64_t* bars = reinterpret_cast<uint64_t*>(sBias + ((plan.bias_floats + 3) & ~3));
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 4);
  const uint32_t bar_a[2] = {smem_u32(bars + 0), smem_u32(bars + 1)};
  const uint32_t bar_d[2] = {smem_u32(bars + 2), smem_u32(bars + 3)};

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int64_t n_gblocks = (a.n + kRows - 1) / kRows;
  const int64_t total_tiles = n_gblocks * a.n_lights;  // tile = gblock * n_lights + light

  // ---- prologue: weights + biases to smem, barriers, TMEM -------------------------------------
  for (int i = tid * 16; i < plan.blob_bytes; i += kMlpThreads * 16)
    *reinterpret_cast<uint4*>(sW + i) = *reinterpret_cast<const uint4*>(a.blob + i);
  for (int i = tid; i < plan.bias_floats; i += kMlpThreads) sBias[i] = a.bias[i];
  if (tid == 0) {
    mbar_init(bar_a[0], kRows);
    mbar_init(bar_a[1], kRows);
    mbar_init(bar_d[0], 1);
    mbar_init(bar_d[1], 1);
    fence_barrier_init();
  }
  if (warp == 8) tmem_alloc(smem_u32(tmem_slot), 2 * kSlotCols);
  fence_proxy_async();  // weights were written with generic stores; UMMA reads via the async proxy
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 8) {
    // ===================== MMA issuer =====================
    uint32_t pa[2] = {0, 0};
    for (int64_t jp = 0;; jp += 2) {
      const bool have0 = blockIdx.x + jp * gridDim.x < total_tiles;
      const bool have1 = blockIdx.x + (jp + 1) * gridDim.x < total_tiles;
      if (!have0) break;
      for (int s = 0; s < plan.n_stages; ++s) {
        const MlpStage& st = plan.st[s];
        const uint32_t idesc = make_idesc(st.n_pad);
        const uint32_t w_addr = smem_u32(sW + st.w_off);
        const int ksteps = st.k_pad >> 4;
        for (int slot = 0; slot < 2; ++slot) {
          if (slot == 1 && !have1) continue;
          mbar_wait(bar_a[slot], pa[slot]);
          pa[slot] ^= 1u;
          tc_fence_after();
          if (lane == 0) {
            const uint32_t a_addr = smem_u32(sA[slot]);
            const uint32_t d_addr = tmem_base + slot * kSlotCols;
            for (int ks = 0; ks < ksteps; ++ks) {
              const int kb = ks >> 2, kin = ks & 3;
              const uint64_t da = make_desc(a_addr + kb * kKBlockBytes + kin * 32);
              const uint64_t db = make_desc(w_addr + kb * (st.n_pad * 128) + kin * 32);
              umma_bf16(d_addr, da, db, idesc, ks > 0 ? 1u : 0u);
            }
            umma_commit(bar_d[slot]);  // arrives when the MMAs above have completed
          }
          __syncwarp();
        }
      }
    }
  } else {
    // ===================== input assembly + epilogue warps =====================
    const int slot = warp >> 2;                 // warps 0-3 -> slot 0, 4-7 -> slot 1
    const int r = (warp & 3) * 32 + lane;       // row of the tile = TMEM lane
    const uint32_t taddr = tmem_base + slot * kSlotCols + ((uint32_t)((warp & 3) * 32) << 16);
    uint8_t* A = sA[slot];
    uint32_t pd = 0;
    for (int64_t j = slot;; j += 2) {
      const int64_t tile = blockIdx.x + j * gridDim.x;
      if (tile >= total_tiles) break;
      const int64_t gblock = tile / a.n_lights;
      const int light = (int)(tile % a.n_lights);
      const int64_t g_raw = gblock * kRows + r;
      const bool row_ok = g_raw < a.n;
      const int64_t g = row_ok ? g_raw : a.n - 1;

      assemble_row(a, g, a.lights.l[light], A, r);
      fence_proxy_async();
      mbar_arrive(bar_a[slot]);

      float sss_keep[3] = {0.f, 0.f, 0.f};
      for (int s = 0; s < plan.n_stages; ++s) {
        const MlpStage& st = plan.st[s];
        const float* bias = sBias + st.b_off;
        mbar_wait(bar_d[slot], pd);
        pd ^= 1u;
        tc_fence_after();
        float v[16];
        if (st.type == ST_HIDDEN || st.type == ST_HEAD_SPLIT_A) {
          // activated columns [0, n_act) -> bf16 -> next stage's A operand
          for (int c0 = 0; c0 < st.n_act; c0 += 16) {
            tmem_ld16(taddr + c0, v);
#pragma unroll
            for (int i = 0; i < 16; ++i) v[i] = act_fn(v[i] + bias[c0 + i], plan.activation, plan.leaky_slope);
            const uint4 lo = make_uint4(pack_bf16(v[0], v[1]), pack_bf16(v[2], v[3]), pack_bf16(v[4], v[5]), pack_bf16(v[6], v[7]));
            const uint4 hi = make_uint4(pack_bf16(v[8], v[9]), pack_bf16(v[10], v[11]), pack_bf16(v[12], v[13]), pack_bf16(v[14], v[15]));
            *reinterpret_cast<uint4*>(A + swz_off(r, (c0 >> 3), kKBlockBytes)) = lo;
            *reinterpret_cast<uint4*>(A + swz_off(r, (c0 >> 3) + 1, kKBlockBytes)) = hi;
          }
          if (st.type == ST_HEAD_SPLIT_A) {  // SSS logits sit right after the activated columns
            tmem_ld16(taddr + st.n_act, v);
#pragma unroll
            for (int c = 0; c < 3; ++c) sss_keep[c] = 1.f / (1.f + __expf(-(v[c] + bias[st.n_act + c])));
          }
          tc_fence_before();
          fence_proxy_async();
          mbar_arrive(bar_a[slot]);
        } else {
          tmem_ld16(taddr, v);
          float4 o;
          if (st.type == ST_HEAD_JOINT) {
            o.x = 1.f / (1.f + __expf(-(v[0] + bias[0])));
            o.y = 1.f / (1.f + __expf(-(v[1] + bias[1])));
            o.z = 1.f / (1.f + __expf(-(v[2] + bias[2])));
            o.w = fmaxf(0.f, v[3] + bias[3]);
          } else {  // ST_HEAD_SPLIT_B
            o = make_float4(sss_keep[0], sss_keep[1], sss_keep[2], fmaxf(0.f, v[0] + bias[0]));
          }
          if (row_ok) {
            a.out_internal[(size_t)g * a.n_lights + light] = o;
            if (a.out_user)
              *reinterpret_cast<float4*>(a.out_user + (int64_t)light * a.user_light_stride + g * 4) = o;
          }
          tc_fence_before();  // TMEM reads are ordered before the next tile's a_ready arrive
        }
      }
    }
  }

  // ---- teardown ----------------------------------------------------------------------------------
  tc_fence_before();
  __syncthreads();
  if (warp == 8) tmem_dealloc(tmem_base, 2 * kSlotCols);
}

}  // namespace

int mlp_smem_bytes(const MlpPlan& plan) {
  return plan.blob_bytes + 2 * plan.max_k_bytes + ((plan.bias_floats + 3) & ~3) * 4 + 4 * 8 + 16 + 1024;
}

int launch_mlp_pack(const sssgs_mlp& mlp, const MlpPlan& plan, uint8_t* blob, float* bias,
                    cudaStream_t s) {
  mlp_pack_kernel<<<32, 256, 0, s>>>(plan, mlp.params, mlp.dtype, blob, bias);
  return 1;
}

int launch_mlp(const sssgs_gaussians& g, const MlpPlan& plan, const uint8_t* blob,
               const float* bias, const CamParams& cam, const LightBatch& lights, int n_lights,
               float4* out_internal, float* out_user, int64_t user_light_stride, int num_sms,
               cudaStream_t s) {
  if (g.n == 0 || n_lights == 0) return 0;
  MlpArgs a;
  a.n = g.n;
  a.means = g.means; a.normals = g.normals; a.rotations = g.rotations; a.scales = g.scales;
  a.vis_sh = g.vis_sh; a.feat = g.feat;
  a.sh_coefs = (g.vis_sh_degree + 1) * (g.vis_sh_degree + 1);
  for (int k = 0; k < 3; ++k) a.cam_pos[k] = cam.pos[k];
  a.lights = lights;
  a.n_lights = n_lights;
  a.blob = blob; a.bias = bias;
  a.out_internal = out_internal; a.out_user = out_user; a.user_light_stride = user_light_stride;
  a.plan = plan;
  const int smem = mlp_smem_bytes(plan);
  static int configured_smem = 0;
  if (smem > configured_smem) {
    if (cudaFuncSetAttribute(mlp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess)
      return -1;
    configured_smem = smem;
  }
  const int64_t tiles = ((g.n + kRows - 1) / kRows) * n_lights;
  const int grid = (int)(tiles < num_sms ? tiles : num_sms);
  mlp_kernel<<<grid, kMlpThreads, smem, s>>>(a);
  return 1;
}

}  // namespace sssgs

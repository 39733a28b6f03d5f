// Joint SSS / incident-light MLP on the 5th-generation tensor cores (hot-path steps a1 + a2).
//
// (L_SSS, L_in) = f_Theta(mu, Sigma, n, w_in, w_out, v) evaluated per Gaussian for a given view
// and point light (Eq. 6; widths and input list L347).  It is a dense batched
// contraction [rows x K] . [K x N] per layer, so it runs as tcgen05.mma (bf16 x bf16 -> fp32):
//
//   * persistent CTAs, one per SM; ALL layer weights live in shared memory for the whole kernel
//     as UMMA operands (K-major, 128-byte swizzle), packed once per call by mlp_pack_kernel;
//   * a row tile = 128 Gaussians x 1 light = the M of one tcgen05.mma (cta_group::1, M=128);
//     its fp32 accumulator [128 x N] sits in TMEM;
//   * up to 4 tiles are in flight per CTA ("slots", 4 or 8 warps each).  A slot is a serial
//     chain  A operand -> MMAs of the layer -> epilogue -> next layer's A operand ; the slots run
//     out of phase so that one slot's epilogue (tcgen05.ld -> bias -> activation -> bf16) runs
//     under the other slots' MMAs.  Activations never touch HBM;
//   * the A operand of a layer is written by the epilogue warps either into shared memory in the
//     UMMA swizzled layout (SS mode: 4 slots when the tiles fit next to the weights) or into
//     TMEM behind the accumulator (TS mode, tcgen05.mma with A from tensor memory: nets whose
//     weights fill shared memory; 2 slots x 8 warps) -- see mlp_shape();
//   * the layer-0 A operand is COMPUTED, not loaded: the same warps assemble the 40+F inputs
//     (unit directions, light distance, SH visibility, Fourier encoding of mu) in fp32 and store
//     them as bf16; a slot walks all lights of a block of 128 Gaussians so that the
//     light-independent inputs are assembled once;
//   * there is no dedicated MMA warp: the first warp of a slot waits for its slot's a_ready
//     mbarrier (all rows written) and one elected lane issues the layer's K steps and commits
//     them to the slot's d_ready mbarrier.
//
// Output: float4 (L_SSS rgb, L_in) per (Gaussian, light), 16 B per row.
#include <cuda_bf16.h>

#include <cstdlib>

#include "internal.cuh"

namespace sssgs {

namespace {

constexpr int kRows = 128;             // rows per tile = UMMA M
constexpr int kKBlockBytes = kRows * 128;  // one 64-wide K block of an smem A tile (128 rows x 128 B)
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
// Instruction descriptor: D = F32, A and B both BF16 (format 1) or both F16 (format 0), both K-major,
// M = 128, N = n.
__device__ __forceinline__ uint32_t make_idesc(int n, bool f16) {
  const uint32_t ab = f16 ? 0u : ((1u << 7) | (1u << 10));
  return (1u << 4) | ab | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(kRows >> 4) << 24);
}

__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
  __nv_bfloat162 h = __floats2bfloat162_rn(a, b);  // .x = a (low half), .y = b
  return *reinterpret_cast<uint32_t*>(&h);
}
// binary16 pair, round to nearest even, finite overflow saturates to +-65504
__device__ __forceinline__ uint32_t pack_f16(float a, float b) {
  uint32_t d;
  asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(b), "f"(a));
  return d;
}
// the 16-bit type of the tensor-core operands: F16 = binary16 (default), else bf16
template <bool F16>
__device__ __forceinline__ uint32_t pack2(float a, float b) {
  return F16 ? pack_f16(a, b) : pack_bf16(a, b);
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
  const bool f16 = plan.f16 != 0;
  pdl_prologue();
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
      uint4 pk = f16 ? make_uint4(pack_f16(v[0], v[1]), pack_f16(v[2], v[3]), pack_f16(v[4], v[5]), pack_f16(v[6], v[7]))
                     : make_uint4(pack_bf16(v[0], v[1]), pack_bf16(v[2], v[3]), pack_bf16(v[4], v[5]),
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
  int slots;                   // row tiles in flight per CTA (1..4)
  int wps;                     // warps per slot: 4 (one per 32 rows) or 8 (two column halves)
  int slot_cols;               // TMEM columns per slot: accumulator D (then the A operand, TS mode)
  int a_col;                   // TS mode: column offset of the A operand inside a slot
  int a_bytes;                 // SS mode: bytes of one slot's A tile in shared memory
  const uint32_t* rows;        // optional: evaluate only the Gaussians rows[0 .. *row_count)
  const uint32_t* row_count;
  int64_t* rows_out;           // optional: receives the number of rows evaluated (SSSGS_CNT_MLP_ROWS)
  MlpPlan plan;
};

constexpr int kKeepChunks = 5;   // 16-byte input chunks a thread keeps in registers across lights
                                 // (chunk 0 and gamma(mu); the per-Gaussian feature is re-read per light, from L2)

__device__ __forceinline__ float act_fn(float v, int activation, float slope) {
  return v > 0.f ? v : (activation == SSSGS_ACT_LEAKY_RELU ? slope * v : 0.f);
}


template <bool F16>
__device__ __forceinline__ uint4 pack8(const float* v) {
  return make_uint4(pack2<F16>(v[0], v[1]), pack2<F16>(v[2], v[3]), pack2<F16>(v[4], v[5]),
                    pack2<F16>(v[6], v[7]));
}

// Step a1, light-independent part.  Input row layout (S1/S13/S14), in
// 16-byte chunks of 8 bf16:
//   chunk 0: n(3) rot(2) scale(3) | chunk 1: w_in(3) w_out(3) d v | chunks 2-4: gamma(mu)(24) |
//   chunks 5..: feat(F), zero padded to in_pad
// Fills keep[0], keep[2..4] (when this thread owns them: c_begin == 0), mu and w_out.
template <bool F16>
__device__ __forceinline__ void assemble_static(const MlpArgs& a, int64_t g, int c_begin, int c_end,
                                                uint4* keep, float mu[3], float wout[3]) {
  mu[0] = a.means[3 * g]; mu[1] = a.means[3 * g + 1]; mu[2] = a.means[3 * g + 2];
  if (c_begin == 0) {
    const float4 q = reinterpret_cast<const float4*>(a.rotations)[g];
    const float sgn = q.x < 0.f ? -1.f : 1.f;
    keep[0] = make_uint4(pack2<F16>(a.normals[3 * g], a.normals[3 * g + 1]),
                         pack2<F16>(a.normals[3 * g + 2], sgn * q.x),
                         pack2<F16>(sgn * q.y, a.scales[3 * g]),
                         pack2<F16>(a.scales[3 * g + 1], a.scales[3 * g + 2]));
    float wox = a.cam_pos[0] - mu[0], woy = a.cam_pos[1] - mu[1], woz = a.cam_pos[2] - mu[2];
    const float io = 1.f / sqrtf(wox * wox + woy * woy + woz * woz);
    wout[0] = wox * io; wout[1] = woy * io; wout[2] = woz * io;
    // gamma(mu): for k = 0..3: [sin(2^k pi mu_xyz), cos(2^k pi mu_xyz)]; octave 0 by sincospif,
    // the next octaves by the double-angle recurrences (error << the bf16 rounding that follows)
    float ga[24];
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
      float s, c;
      sincospif(mu[ax], &s, &c);
      ga[ax] = s; ga[3 + ax] = c;
#pragma unroll
      for (int k = 1; k < 4; ++k) {
        const float s2 = 2.f * s * c, c2 = 1.f - 2.f * s * s;
        s = s2; c = c2;
        ga[6 * k + ax] = s; ga[6 * k + 3 + ax] = c;
      }
    }
    keep[2] = pack8<F16>(ga);
    keep[3] = pack8<F16>(ga + 8);
    keep[4] = pack8<F16>(ga + 16);
  }
}

// Light-dependent chunk 1: (w_in, w_out, d, v) for light `lt`.
template <bool F16>
__device__ __forceinline__ uint4 assemble_light(const MlpArgs& a, int64_t g, const LightParams& lt,
                                                const float mu[3], const float wout[3]) {
  float wix = lt.pos[0] - mu[0], wiy = lt.pos[1] - mu[1], wiz = lt.pos[2] - mu[2];
  const float d = sqrtf(wix * wix + wiy * wiy + wiz * wiz);
  const float id = 1.f / d;
  wix *= id; wiy *= id; wiz *= id;
  float v;
  if (a.sh_coefs == 4) {
    const float4 sh = reinterpret_cast<const float4*>(a.vis_sh)[g];
    v = kY00 * sh.x + kY1 * (sh.y * wiy + sh.z * wiz + sh.w * wix);
  } else {
    v = kY00 * a.vis_sh[g];
  }
  v = fminf(1.f, fmaxf(0.f, v));
  return make_uint4(pack2<F16>(wix, wiy), pack2<F16>(wiz, wout[0]), pack2<F16>(wout[1], wout[2]),
                    pack2<F16>(d, v));
}

// ---- TMEM helpers ---------------------------------------------------------------------------------
// The A operand of every layer lives in TMEM (tcgen05.mma with A from tensor memory): row m of the
// tile is TMEM lane m, and 32-bit column j of the operand holds the bf16 pair (k = 2j, 2j + 1), low
// half first.  Only the weights are read from shared memory by the tensor core.
__device__ __forceinline__ void tmem_st4(uint32_t taddr, uint4 v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(v.x),
               "r"(v.y), "r"(v.z), "r"(v.w)
               : "memory");
}
__device__ __forceinline__ void tmem_wait_st() {
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
// D[tmem] (+)= A[tmem] . B[smem desc]^T, kind::f16 (bf16 inputs, fp32 accumulate); ACC = false
// overwrites D.  The predicate is a compile-time constant so that the issuing lane spends no
// instructions on it: the K steps of a stage are issued back to back by one thread, and every
// instruction in that loop adds latency between tensor-core dispatches.
template <bool ACC>
__device__ __forceinline__ void umma_bf16_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t desc_b,
                                             uint32_t idesc) {
  if (ACC) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.eq.u32 p, 1, 1;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(tmem_d), "r"(tmem_a), "l"(desc_b), "r"(idesc)
        : "memory");
  } else {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.eq.u32 p, 1, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(tmem_d), "r"(tmem_a), "l"(desc_b), "r"(idesc)
        : "memory");
  }
}

// Same with A from shared memory (K-major, 128-byte swizzle descriptors for both operands).
template <bool ACC>
__device__ __forceinline__ void umma_bf16_ss(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b,
                                             uint32_t idesc) {
  if (ACC) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.eq.u32 p, 1, 1;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc)
        : "memory");
  } else {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.eq.u32 p, 1, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc)
        : "memory");
  }
}
__device__ __forceinline__ void sts128(uint32_t saddr, uint4 v) {
  asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(saddr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w)
               : "memory");
}

// Where one thread writes its row of a slot's A operand.  Two modes (template flag TS):
//   TS: A in TMEM at `at` (this thread's lane; 16-byte chunk c = columns at + 4c .. 4c + 3)
//   SS: A in shared memory, K-major with the 128-byte swizzle: chunk c of the row sits at
//       rowbase + (c / 8) * kKBlockBytes + (((c % 8) << 4) ^ swz), swz = (row % 8) << 4
struct ARow {
  uint32_t at, rowbase, swz;
};
template <bool TS>
__device__ __forceinline__ void a_store(const ARow& ar, int c, uint4 v) {
  if (TS) tmem_st4(ar.at + 4 * c, v);
  else sts128(ar.rowbase + (uint32_t)(c >> 3) * (uint32_t)kKBlockBytes + ((((uint32_t)c & 7u) << 4) ^ ar.swz), v);
}
// Makes this thread's A-operand writes visible to the tensor core before it signals a_ready.
template <bool TS>
__device__ __forceinline__ void a_publish() {
  if (TS) {
    tmem_wait_st();
    tc_fence_before();
  } else {
    tc_fence_before();
    fence_proxy_async();
  }
}

// Writes the 16-byte chunks [c_begin, c_end) of this thread's row of the layer-0 A operand.
template <bool TS, bool F16>
__device__ __forceinline__ void write_row(const MlpArgs& a, int64_t g, const ARow& ar, int c_begin,
                                          int c_end, const uint4* keep, const uint4& light_chunk) {
#pragma unroll
  for (int c = 0; c < kKeepChunks; ++c)
    if (c >= c_begin && c < c_end) a_store<TS>(ar, c, (c == 1) ? light_chunk : keep[c]);
  // the per-Gaussian feature (chunks 5..) is read here: it stays L2-resident across the lights
  const int F = a.plan.feat_dim;
  for (int c = max(c_begin, kKeepChunks); c < c_end; ++c) {
    const int j = (c - 5) * 8;
    float4 f0 = make_float4(0.f, 0.f, 0.f, 0.f), f1 = f0;
    if (j < F) f0 = *reinterpret_cast<const float4*>(a.feat + g * F + j);
    if (j + 4 < F) f1 = *reinterpret_cast<const float4*>(a.feat + g * F + j + 4);
    a_store<TS>(ar, c, make_uint4(pack2<F16>(f0.x, f0.y), pack2<F16>(f0.z, f0.w), pack2<F16>(f1.x, f1.y),
                                  pack2<F16>(f1.z, f1.w)));
  }
}

// ---- epilogue helpers --------------------------------------------------------------------------
// 16 accumulator columns of this thread's row, TMEM -> registers, asynchronously: the registers
// are valid only after tmem_wait16 on the same array (which carries the data dependence).
__device__ __forceinline__ void tmem_ld16_async(uint32_t taddr, uint32_t* r) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]),
        "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]),
        "=r"(r[14]), "=r"(r[15])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_wait16(uint32_t* r) {
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
  // empty volatile asms keep their order after the wait and make every later use of r[i] depend on it
#pragma unroll
  for (int i = 0; i < 16; ++i) asm volatile("" : "+r"(r[i]));
}
// 16-bit pair {lo, hi} = round-to-nearest-even of (max(lo, 0), max(hi, 0)): the ReLU rides on the convert
template <bool F16>
__device__ __forceinline__ uint32_t pack2_relu(float lo, float hi) {
  uint32_t d;
  if (F16) asm("cvt.rn.relu.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  else asm("cvt.rn.relu.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}
// (x0, x1) += (y0, y1) as one packed fp32x2 add (sm_100 FADD2)
__device__ __forceinline__ void add2(float& x0, float& x1, float y0, float y1) {
  asm("{\n\t.reg .b64 a, b;\n\t"
      "mov.b64 a, {%0, %1};\n\t"
      "mov.b64 b, {%2, %3};\n\t"
      "add.rn.f32x2 a, a, b;\n\t"
      "mov.b64 {%0, %1}, a;\n\t}"
      : "+f"(x0), "+f"(x1)
      : "f"(y0), "f"(y1));
}
// 16 bias values from shared memory.  Not volatile: the biases never change during the kernel, so
// the compiler may schedule these loads ahead of the TMEM wait they are independent of.
__device__ __forceinline__ void lds_bias16(uint32_t saddr, float4* b) {
#pragma unroll
  for (int q = 0; q < 4; ++q)
    asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
        : "=f"(b[q].x), "=f"(b[q].y), "=f"(b[q].z), "=f"(b[q].w)
        : "r"(saddr + 16u * q));
}

// bias + activation + bf16 of the 16 accumulator columns c0 .. c0 + 15 -> next A operand.
template <bool RELU, bool TS, bool F16>
__device__ __forceinline__ void finish16(const uint32_t* r, const float4* b, const ARow& ar, int c0,
                                         int activation, float slope) {
  float v[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    add2(v[4 * q], v[4 * q + 1], b[q].x, b[q].y);
    add2(v[4 * q + 2], v[4 * q + 3], b[q].z, b[q].w);
  }
  uint32_t w[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    if (RELU) {
      w[i] = pack2_relu<F16>(v[2 * i], v[2 * i + 1]);
    } else {
      w[i] = pack2<F16>(act_fn(v[2 * i], activation, slope), act_fn(v[2 * i + 1], activation, slope));
    }
  }
  a_store<TS>(ar, c0 >> 3, make_uint4(w[0], w[1], w[2], w[3]));
  a_store<TS>(ar, (c0 >> 3) + 1, make_uint4(w[4], w[5], w[6], w[7]));
}

// Hidden-stage epilogue of one thread: its share of the activated columns [0, n_act), in groups
// of 16, with the TMEM load of the next group in flight while the current one is finished.
// WPS = 4: all columns; WPS = 8: the two warps of a row quarter take alternate 32-column blocks.
// d_taddr: this thread's lane base in the slot's accumulator.
template <int WPS_, bool RELU, bool TS, bool F16>
__device__ __forceinline__ void hidden_epilogue(uint32_t d_taddr, const ARow& ar, uint32_t bias_saddr,
                                                int n_act, int half, int activation, float slope) {
  constexpr int G = WPS_ == 4 ? 8 : 4;  // groups of 16 columns per thread for 128 columns
  uint32_t ra[16], rb[16];
  float4 ba[4], bb[4];
  // group gi covers columns col(gi) .. +15
  auto col = [&](int gi) { return WPS_ == 4 ? 16 * gi : 32 * half + 64 * (gi >> 1) + 16 * (gi & 1); };
  if (col(0) + 16 <= n_act) tmem_ld16_async(d_taddr + col(0), ra);
#pragma unroll
  for (int gp = 0; gp < G / 2; ++gp) {
    const int c0 = col(2 * gp), c1 = col(2 * gp + 1);
    if (c0 + 16 > n_act) break;
    lds_bias16(bias_saddr + 4u * c0, ba);
    tmem_wait16(ra);
    if (c1 + 16 <= n_act) tmem_ld16_async(d_taddr + c1, rb);
    finish16<RELU, TS, F16>(ra, ba, ar, c0, activation, slope);
    if (c1 + 16 > n_act) break;
    lds_bias16(bias_saddr + 4u * c1, bb);
    tmem_wait16(rb);
    if (2 * gp + 2 < G) {
      const int c2 = col(2 * gp + 2);
      if (c2 + 16 <= n_act) tmem_ld16_async(d_taddr + c2, ra);
    }
    finish16<RELU, TS, F16>(rb, bb, ar, c1, activation, slope);
  }
}

constexpr int kMaxSlots = 4;

#ifdef SSSGS_MLP_TIMELINE
// Debug builds only (-DSSSGS_MLP_TIMELINE): SM-clock stamps of one CTA's slots, read back with
// sssgs_debug_mlp_timeline().  Not compiled into the product library.
__device__ long long g_timeline[kMaxSlots][512];
#define TL_STAMP(code)                                                              \
  do {                                                                              \
    if (blockIdx.x == 0 && wq == 0 && lane == 0 && tl_n < 510) {                    \
      g_timeline[slot][tl_n++] = (clock64() << 4) | (code);                         \
      g_timeline[slot][511] = tl_n;                                                 \
    }                                                                               \
  } while (0)
#else
#define TL_STAMP(code) do {} while (0)
#endif
constexpr int kMlpThreadsMax = 512;  // up to 16 warps: 4 slots x 4 warps or 2 slots x 8 warps

// Work distribution: a "unit" is a block of 128 Gaussians with all the lights of the batch; slot s of
// CTA b owns the units (i * slots + s) * gridDim.x + b, i = 0, 1, ...  Within a unit the lights are
// walked in order so that the light-independent inputs of a row are assembled once.
template <int WPS, bool RELU, bool TS, bool F16>
__global__ void __launch_bounds__(kMlpThreadsMax, 1) mlp_kernel(const __grid_constant__ MlpArgs a) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  const MlpPlan& plan = a.plan;
  const int S = a.slots;
  uint8_t* sW = smem;
  uint8_t* sA0 = smem + plan.blob_bytes;  // SS mode: one A tile per slot (a_bytes = 0 in TS mode)
  float* sBias = reinterpret_cast<float*>(sA0 + S * a.a_bytes);
  uint64_t* bars = reinterpret_cast<uint64_t*>(sBias + ((plan.bias_floats + 3) & ~3));
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * kMaxSlots);
  uint32_t* issue_lock = tmem_slot + 1;  // serialises the slots' MMA batches (see issue_stage)
  // bars[s] = a_ready of slot s, bars[kMaxSlots + s] = d_ready of slot s

  pdl_prologue();
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int64_t n_rows = a.rows ? (int64_t)*a.row_count : a.n;
  // A unit = 128 rows x a range of the batch's lights.  All lights when there are plenty of row
  // blocks (the light-independent inputs are then assembled once per block); with few blocks the
  // lights are split so that every slot of every CTA gets about 3 units or more.
  const int64_t n_blocks = (n_rows + kRows - 1) / kRows;
  int split = 1;
  while (split < a.n_lights && n_blocks * split < 3ll * S * gridDim.x) split *= 2;
  if (split > a.n_lights) split = a.n_lights;
  const int lights_per_unit = (a.n_lights + split - 1) / split;
  split = (a.n_lights + lights_per_unit - 1) / lights_per_unit;
  const int64_t n_units = n_blocks * split;
  if (a.rows_out && blockIdx.x == 0 && threadIdx.x == 0) *a.rows_out = n_rows;

  // ---- prologue: weights + biases to smem, barriers, TMEM -------------------------------------
  for (int i = tid * 16; i < plan.blob_bytes; i += blockDim.x * 16)
    *reinterpret_cast<uint4*>(sW + i) = *reinterpret_cast<const uint4*>(a.blob + i);
  for (int i = tid; i < plan.bias_floats; i += blockDim.x) sBias[i] = a.bias[i];
  if (tid == 0) {
    for (int s = 0; s < S; ++s) {
      mbar_init(smem_u32(bars + s), WPS * 32);
      mbar_init(smem_u32(bars + kMaxSlots + s), 1);
    }
    *issue_lock = 0u;
    fence_barrier_init();
  }
  if (warp == 0) tmem_alloc(smem_u32(tmem_slot), 512);
  fence_proxy_async();  // weights were written with generic stores; UMMA reads via the async proxy
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  {
    // ===================== input assembly + epilogue warps =====================
    // a warp may only touch the TMEM lanes 32 * (warp % 4) .. +31: WPS is 4 or 8, so warp % 4 is
    // also the row quarter inside the slot
    const int slot = warp / WPS, wq = warp % WPS;
    const int quarter = wq & 3, half = wq >> 2;   // column half (WPS = 8)
    const int r = quarter * 32 + lane;            // row of the tile = TMEM lane
    // this thread's lane base in the slot's accumulator (d) and A operand (at)
    const uint32_t taddr = tmem_base + slot * a.slot_cols + ((uint32_t)(quarter * 32) << 16);
    ARow ar;
    ar.at = taddr + a.a_col;
    ar.rowbase = smem_u32(sA0 + slot * a.a_bytes) + (uint32_t)(r * 128);
    ar.swz = (uint32_t)((r & 7) << 4);
    const uint32_t bar_a = smem_u32(bars + slot), bar_d = smem_u32(bars + kMaxSlots + slot);
    // The first warp of a slot also issues the slot's MMAs: once all rows of the A operand have
    // arrived (a_ready), one elected lane issues the K steps of the stage and commits them to
    // d_ready.  A slot's pipeline is serial anyway (A operand -> MMA -> epilogue -> next A operand);
    // the tensor core is kept busy by the other slots.
    int tl_n = 0;
    (void)tl_n;
    uint32_t pa = 0;
    auto issue_stage = [&](int s_idx) {
      if (wq != 0) return;
      TL_STAMP(0);
      mbar_wait(bar_a, pa);
      pa ^= 1u;
      tc_fence_after();
      TL_STAMP(1);
      if (lane == 0) {
        // TS mode (two slots): one slot's K steps go to the tensor core as a batch.  If the two slots
        // interleaved their steps they would finish together and stay in lock-step (both in the
        // epilogue, then both waiting for the tensor core); batching staggers them so that one
        // slot's epilogue runs under the other's MMAs.
        if (TS) {
          while (atomicCAS(issue_lock, 0u, 1u) != 0u) {
          }
        }
        TL_STAMP(6);
        const MlpStage& st = plan.st[s_idx];
        const uint32_t idesc = make_idesc(st.n_pad, F16);
        const uint32_t w_addr = smem_u32(sW + st.w_off);
        const uint32_t d_addr = tmem_base + slot * a.slot_cols;
        const uint32_t a_addr = d_addr + a.a_col;                          // TS: A operand in TMEM
        const uint32_t a_smem = smem_u32(sA0 + slot * a.a_bytes);          // SS: A tile in smem
        // one K step = 16 bf16 = 8 TMEM columns of A and 32 bytes inside a 128-byte swizzled row of
        // the weights (the descriptor's start address advances by 32 >> 4; the second 64-wide K block
        // starts n_pad * 128 bytes further)
        const int ksteps = st.k_pad >> 4;
        const uint64_t db0 = make_desc(w_addr);
        const uint64_t db1 = make_desc(w_addr + st.n_pad * 128);
        if (TS) {
          umma_bf16_ts<false>(d_addr, a_addr, db0, idesc);
#pragma unroll
          for (int ks = 1; ks < 8; ++ks)
            if (ks < ksteps) umma_bf16_ts<true>(d_addr, a_addr + ks * 8, (ks < 4 ? db0 : db1) + (uint64_t)((ks & 3) * 2), idesc);
        } else {
          const uint64_t da0 = make_desc(a_smem), da1 = make_desc(a_smem + kKBlockBytes);
          umma_bf16_ss<false>(d_addr, da0, db0, idesc);
#pragma unroll
          for (int ks = 1; ks < 8; ++ks)
            if (ks < ksteps)
              umma_bf16_ss<true>(d_addr, (ks < 4 ? da0 : da1) + (uint64_t)((ks & 3) * 2),
                                 (ks < 4 ? db0 : db1) + (uint64_t)((ks & 3) * 2), idesc);
        }
        umma_commit(bar_d);  // arrives when the MMAs above have completed
        if (TS) atomicExch(issue_lock, 0u);
      }
      __syncwarp();
      TL_STAMP(2);
    };
    // 16-byte input chunks this thread writes
    const int nchunks = plan.in_pad >> 3;
    const int c_split = nchunks > 5 ? 5 : nchunks;
    const int c_begin = (WPS == 8 && half == 1) ? c_split : 0;
    const int c_end = (WPS == 8 && half == 0) ? c_split : nchunks;
    uint32_t pd = 0;
    for (int64_t u = (int64_t)slot * gridDim.x + blockIdx.x; u < n_units; u += (int64_t)S * gridDim.x) {
      const int64_t row = (u / split) * kRows + r;
      const int light0 = (int)(u % split) * lights_per_unit;
      const int light1 = min(a.n_lights, light0 + lights_per_unit);
      const bool row_ok = row < n_rows;
      const int64_t row_c = row_ok ? row : n_rows - 1;
      const int64_t g = a.rows ? (int64_t)a.rows[row_c] : row_c;
      uint4 keep[kKeepChunks];
      float mu[3], wout[3];
      assemble_static<F16>(a, g, c_begin, c_end, keep, mu, wout);
      for (int light = light0; light < light1; ++light) {
        uint4 lc = make_uint4(0u, 0u, 0u, 0u);
        if (c_begin == 0) lc = assemble_light<F16>(a, g, a.lights.l[light], mu, wout);
        write_row<TS, F16>(a, g, ar, c_begin, c_end, keep, lc);
        a_publish<TS>();
        mbar_arrive(bar_a);
        issue_stage(0);

        float sss_keep[3] = {0.f, 0.f, 0.f};
        for (int s = 0; s < plan.n_stages; ++s) {
          const MlpStage& st = plan.st[s];
          const float* bias = sBias + st.b_off;
          mbar_wait(bar_d, pd);
          pd ^= 1u;
          tc_fence_after();
          TL_STAMP(3);
          if (st.type == ST_HIDDEN || st.type == ST_HEAD_SPLIT_A) {
            // activated columns [0, n_act) -> bf16 -> next stage's A operand
            hidden_epilogue<WPS, RELU, TS, F16>(taddr, ar, smem_u32(bias), st.n_act, half, plan.activation, plan.leaky_slope);
            if (st.type == ST_HEAD_SPLIT_A && half == 0) {  // SSS logits sit right after the activated columns
              float v[16];
              tmem_ld16(taddr + st.n_act, v);
#pragma unroll
              for (int c = 0; c < 3; ++c) sss_keep[c] = 1.f / (1.f + __expf(-(v[c] + bias[st.n_act + c])));
            }
            TL_STAMP(4);
            a_publish<TS>();
            mbar_arrive(bar_a);
            issue_stage(s + 1);
          } else {
            if (half == 0) {
              float v[16];
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
            }
            TL_STAMP(5);
            tc_fence_before();  // TMEM reads are ordered before the next tile's a_ready arrive
          }
        }
      }
    }
  }

  // ---- teardown ----------------------------------------------------------------------------------
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem_base, 512);
}

}  // namespace

// How a plan runs.  A slot (one 128-row tile in flight) needs its fp32 accumulator in TMEM (widest
// layer, rounded up to 32 columns) and its bf16 A operand either in shared memory (SS mode: one
// max_k_bytes tile per slot next to the weights) or in TMEM behind the accumulator (TS mode: widest
// input / 2 columns).  Reading accumulators back is the binding resource (TMEM reads ~64 B/clk per
// SM), and TS mode adds the A reads to it, so SS mode is used whenever shared memory
// holds 4 tiles (or more tiles than TMEM would); wide nets whose weights fill shared memory run in
// TS mode.  At most 4 slots (512 TMEM columns, 16 warps).
struct MlpShape {
  int slots, wps, slot_cols, a_col, a_bytes;
  bool ts;
};
static MlpShape mlp_shape(const MlpPlan& plan) {
  const int d_cols = (plan.max_n + 31) / 32 * 32;
  const int a_cols = plan.max_k_bytes / (kRows * 128) * 32;  // K blocks of 64 bf16 = 32 columns each
  const int fixed = plan.blob_bytes + ((plan.bias_floats + 3) & ~3) * 4 + 2 * kMaxSlots * 8 + 16 + 1024;
  int s_ss = (227 * 1024 - fixed) / plan.max_k_bytes;
  if (s_ss > 512 / d_cols) s_ss = 512 / d_cols;
  if (s_ss > kMaxSlots) s_ss = kMaxSlots;
  int s_ts = 512 / (d_cols + a_cols);
  if (s_ts > kMaxSlots) s_ts = kMaxSlots;
  MlpShape sh;
  sh.ts = !(s_ss >= kMaxSlots || s_ss > s_ts);
  sh.slots = sh.ts ? s_ts : s_ss;
  if (sh.slots < 1) sh.slots = 1;
  sh.wps = sh.slots <= 2 ? 8 : 4;
  {  // tuning aid: SSSGS_MLP_SHAPE=<ts><slots><wps>, e.g. 124 = TS mode, 2 slots, 4 warps per slot
    static int force = -1;
    if (force < 0) { const char* e = getenv("SSSGS_MLP_SHAPE"); force = e ? atoi(e) : 0; }
    if (force > 0) {
      const bool ts = force / 100 != 0;
      const int slots = force / 10 % 10, wps = force % 10;
      if (slots >= 1 && slots <= (ts ? s_ts : s_ss) && (wps == 4 || wps == 8)) {
        sh.ts = ts; sh.slots = slots; sh.wps = wps;
      }
    }
  }
  sh.slot_cols = sh.ts ? d_cols + a_cols : d_cols;
  sh.a_col = d_cols;
  sh.a_bytes = sh.ts ? 0 : plan.max_k_bytes;
  return sh;
}

int mlp_smem_bytes(const MlpPlan& plan) {
  const MlpShape sh = mlp_shape(plan);
  return plan.blob_bytes + sh.slots * sh.a_bytes + ((plan.bias_floats + 3) & ~3) * 4 + 2 * kMaxSlots * 8 + 16 + 1024;
}

int launch_mlp_pack(const sssgs_mlp& mlp, const MlpPlan& plan, uint8_t* blob, float* bias,
                    cudaStream_t s) {
  launch_pdl(mlp_pack_kernel, dim3(32), dim3(256), 0, s, plan, mlp.params, mlp.dtype, blob, bias);
  return 1;
}

int launch_mlp(const sssgs_gaussians& g, const MlpPlan& plan, const uint8_t* blob,
               const float* bias, const CamParams& cam, const LightBatch& lights, int n_lights,
               float4* out_internal, float* out_user, int64_t user_light_stride, int max_ctas,
               const uint32_t* rows, const uint32_t* row_count, int64_t* rows_out, cudaStream_t s) {
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
  a.rows = rows; a.row_count = row_count; a.rows_out = rows_out;
  const MlpShape sh = mlp_shape(plan);
  a.slots = sh.slots; a.wps = sh.wps; a.slot_cols = sh.slot_cols; a.a_col = sh.a_col; a.a_bytes = sh.a_bytes;
  const int smem = mlp_smem_bytes(plan);
  const int64_t units = (g.n + kRows - 1) / kRows;
  int grid = (int)(units < max_ctas ? units : max_ctas);
  {  // tuning aid: SSSGS_MLP_SMS caps the number of CTAs (= SMs) the MLP occupies
    static int cap = -1;
    if (cap < 0) { const char* e = getenv("SSSGS_MLP_SMS"); cap = e ? atoi(e) : 0; }
    if (cap > 0 && grid > cap) grid = cap;
  }
  const bool relu = plan.activation == SSSGS_ACT_RELU;
  auto launch = [&](auto kernel) -> int {
    if (ensure_dyn_smem(reinterpret_cast<const void*>(kernel), smem) != cudaSuccess) return -1;
    launch_pdl(kernel, dim3(grid), dim3(a.slots * a.wps * 32), (size_t)smem, s, a);
    return 1;
  };
  const int v = (plan.f16 ? 8 : 0) + (a.wps == 8 ? 4 : 0) + (relu ? 2 : 0) + (sh.ts ? 1 : 0);
  switch (v) {
    case 0: return launch(mlp_kernel<4, false, false, false>);
    case 1: return launch(mlp_kernel<4, false, true, false>);
    case 2: return launch(mlp_kernel<4, true, false, false>);
    case 3: return launch(mlp_kernel<4, true, true, false>);
    case 4: return launch(mlp_kernel<8, false, false, false>);
    case 5: return launch(mlp_kernel<8, false, true, false>);
    case 6: return launch(mlp_kernel<8, true, false, false>);
    case 7: return launch(mlp_kernel<8, true, true, false>);
    case 8: return launch(mlp_kernel<4, false, false, true>);
    case 9: return launch(mlp_kernel<4, false, true, true>);
    case 10: return launch(mlp_kernel<4, true, false, true>);
    case 11: return launch(mlp_kernel<4, true, true, true>);
    case 12: return launch(mlp_kernel<8, false, false, true>);
    case 13: return launch(mlp_kernel<8, false, true, true>);
    case 14: return launch(mlp_kernel<8, true, false, true>);
    default: return launch(mlp_kernel<8, true, true, true>);
  }
}

}  // namespace sssgs

#ifdef SSSGS_MLP_TIMELINE
extern "C" int sssgs_debug_mlp_timeline(long long* out) {
  return (int)cudaMemcpyFromSymbol(out, sssgs::g_timeline, sizeof(long long) * sssgs::kMaxSlots * 512);
}
#endif

// Joint SSS / incident-light MLP on the 5th-generation tensor cores (hot-path steps a1 + a2).
//
// (L_SSS, L_in) = f_Theta(mu, Sigma, n, w_in, w_out, v) evaluated per Gaussian for a given view
// and point light (Eq. 6; widths and input list L347).  It is a dense batched
// contraction [rows x K] . [K x N] per layer, so it runs as tcgen05.mma (16 bit x 16 bit -> fp32):
//
//   * persistent CTAs, one per SM; ALL layer weights live in shared memory for the whole kernel
//     as UMMA B operands (K-major, 128-byte swizzle), packed once per call by mlp_pack_kernel;
//   * a row tile = 128 Gaussians x 1 light = the M of one tcgen05.mma (cta_group::1, M=128);
//     its fp32 accumulator [128 x N] sits in TMEM, and so does the A operand of every layer
//     (tcgen05.mma with A from tensor memory): the epilogue warps write the next layer's input
//     straight back into tensor memory with tcgen05.st.  Activations never touch shared memory or
//     HBM; shared memory only serves the tensor core's reads of the weights (measured: with the A
//     tiles and the biases in shared memory its 128 B/clk, not the tensor core, bound the kernel);
//   * the biases ride on the tensor core too: every stage starts with one extra K step whose A
//     operand is a constant tile of ones (8 TMEM columns, written once per CTA) and whose B operand
//     holds the bias split in three 16-bit terms (b = hi + mid + lo, exact to ~2^-30 |b|), so the
//     accumulator comes out of the MMAs with the bias in it and the epilogue is
//     tcgen05.ld -> activation -> 16-bit convert -> tcgen05.st with no shared-memory loads at all;
//   * up to 4 tiles are in flight per CTA ("slots", 4 or 8 warps each).  A slot is a serial
//     chain  A operand -> MMAs of the layer -> epilogue -> next layer's A operand ; the slots run
//     out of phase so that one slot's epilogue runs under the other slots' MMAs;
//   * the layer-0 A operand is COMPUTED, not loaded: the same warps assemble the 40+F inputs
//     (unit directions, light distance, SH visibility, Fourier encoding of mu) in fp32 and store
//     them as 16-bit values; a slot walks all lights of a block of 128 Gaussians so that the
//     light-independent inputs are assembled once;
//   * there is no dedicated MMA warp: the first warp of a slot waits for its slot's a_ready
//     mbarrier (all rows written) and issues the stage's K steps and the commit to the slot's d_ready
//     mbarrier.  The whole warp runs the issue code with warp-uniform operands and the tcgen05
//     instructions are predicated on one elected lane, so that the operands live in uniform
//     registers: inside a divergent `if (lane == 0)` every operand of every MMA goes through R2UR
//     and one MMA is issued per ~100-115 clocks instead of one per ~70 (profiles/r02_tmem_ld_microbench.md).
//
// Output: float4 (L_SSS rgb, L_in) per (Gaussian, light), 16 B per row.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <cstdlib>
#include <type_traits>

#include "internal.cuh"

namespace sssgs {

namespace {

constexpr int kRows = 128;             // rows per tile = UMMA M
constexpr int kOnesCols = 8;           // TMEM columns of the constant-ones A operand (one K step)
constexpr int kTmemCols = 512;
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
// TMA bulk copy (no tensor map: a linear range), global -> shared, completion counted in bytes on an mbarrier
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_copy_g2s(uint32_t dst_smem, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst_smem),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
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
// value of the low 16-bit half of a packed pair, back in fp32
__device__ __forceinline__ float unpack_lo(uint32_t p, bool f16) {
  if (f16) return __half2float(__ushort_as_half((unsigned short)(p & 0xFFFFu)));
  return __uint_as_float(p << 16);
}
// byte offset of 16-byte chunk `c` (8 x 16 bit = columns 8c..8c+7) of row `r` inside a K-major
// SWIZZLE_128B operand whose 64-column K blocks are `rows*128` bytes apart
__device__ __forceinline__ uint32_t swz_off(int r, int c, int kblock_bytes) {
  return (uint32_t)((c >> 3) * kblock_bytes + r * 128 + (((c & 7) ^ (r & 7)) << 4));
}

// ---------------------------------------------------------------------------------------------
// Weight packer: caller's W[out][in] (+ bias) -> 16-bit UMMA B operands in the swizzled layout.
// Blob = the stages' weights, then the bias blocks: block q holds the biases of stages 4q .. 4q+3,
// stage s in the 16-column K slot s % 4 of a [max_n x 64] K-major tile (the K step an MMA reads is
// selected by the start address of its descriptor, like the K steps of a weight block): row n =
// (hi, mid, lo, 0, ...) with bias[n] = hi + mid + lo in the operand type.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
mlp_pack_kernel(MlpPlan plan, const void* __restrict__ params, int dtype, uint8_t* __restrict__ blob) {
  const bool f16 = plan.f16 != 0;
  pdl_prologue();
  auto load = [&](int off) -> float {
    if (dtype == SSSGS_BF16)
      return __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(params)[off]);
    return reinterpret_cast<const float*>(params)[off];
  };
  auto pack = [&](float a, float b) -> uint32_t { return f16 ? pack_f16(a, b) : pack_bf16(a, b); };
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
      const uint4 pk = make_uint4(pack(v[0], v[1]), pack(v[2], v[3]), pack(v[4], v[5]), pack(v[6], v[7]));
      *reinterpret_cast<uint4*>(blob + st.w_off + swz_off(r, c, st.n_pad * 128)) = pk;
    }
  }
  // bias blocks
  const int n_blks = (plan.n_stages + 3) / 4;
  const int blk_bytes = plan.max_n * 128;
  for (int q = blockIdx.x * 256 + threadIdx.x; q < n_blks * plan.max_n * 8; q += gridDim.x * 256) {
    const int c = q & 7, r = (q >> 3) % plan.max_n, blk = (q >> 3) / plan.max_n;
    const int s = blk * 4 + (c >> 1);
    uint4 pk = make_uint4(0u, 0u, 0u, 0u);
    if ((c & 1) == 0 && s < plan.n_stages && r < plan.st[s].n_pad) {
      const MlpStage& st = plan.st[s];
      float b = 0.f;
      if (r < st.src_rows[0]) b = load(st.src_b[0] + r);
      else if (r < st.src_rows[0] + st.src_rows[1]) b = load(st.src_b[1] + (r - st.src_rows[0]));
      // b = hi + mid + lo: every term is the 16-bit rounding of what is left (the differences are exact in fp32)
      const uint32_t p_hi = pack(b, 0.f);
      const float r1 = b - unpack_lo(p_hi, f16);
      const uint32_t p_mid = pack(r1, 0.f);
      const float r2 = r1 - unpack_lo(p_mid, f16);
      const uint32_t p_lo = pack(r2, 0.f);
      pk = make_uint4((p_hi & 0xFFFFu) | (p_mid << 16), p_lo & 0xFFFFu, 0u, 0u);
    }
    *reinterpret_cast<uint4*>(blob + plan.bias_off + blk * blk_bytes + swz_off(r, c, blk_bytes)) = pk;
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
  float4* out_internal;        // [n][n_lights]
  float* out_user;             // optional: light l at out_user + l*user_light_stride, [n][4]
  int64_t user_light_stride;   // in floats
  int slots;                   // row tiles in flight per CTA (1..4)
  int wps;                     // warps per slot: 4 (one per 32 rows) or 8 (two column halves)
  // TMEM columns (mlp_shape): slot s owns  D = d_stride s,  H = h_base + 16 s,  A = a_base + a_stride s,
  // A0 = a0_base + a0_stride s;  the constant-ones operand sits in the last 8 columns of the allocation
  int d_stride;                // accumulator of the hidden stages (widest layer, 32-column granules)
  int h_base;                  // accumulator of the last stage (16 columns of its own)
  int a_base, a_stride;        // A operand of the hidden layers and the last stage
  int a0_base, a0_stride;      // A operand of layer 0 (its own region: see write_static)
  int stagger;                 // SM clocks by which consecutive slots start apart
  int plain_copy;              // measurement aid: weights copied by all threads instead of TMA bulk copies
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
// 16-byte chunks of 8 x 16 bit:
//   chunk 0: n(3) rot(2) scale(3) | chunk 1: w_in(3) w_out(3) d v | chunks 2-4: gamma(mu)(24) |
//   chunks 5..: feat(F), zero padded to in_pad
// Fills keep[0], keep[2..4] (when this thread owns them: c_begin == 0), mu and w_out.
template <bool F16>
__device__ __forceinline__ void assemble_static(const MlpArgs& a, int64_t g, int c_begin, int c_end,
                                                uint4* keep, float mu[3], float wout[3], float4& sh) {
  mu[0] = a.means[3 * g]; mu[1] = a.means[3 * g + 1]; mu[2] = a.means[3 * g + 2];
  if (c_begin == 0) {
    // visibility SH of the row, kept in registers across the lights of the block
    if (a.sh_coefs == 4) sh = reinterpret_cast<const float4*>(a.vis_sh)[g];
    else sh = make_float4(a.vis_sh[g], 0.f, 0.f, 0.f);
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
    // the next octaves by the double-angle recurrences (error << the 16-bit rounding that follows)
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
__device__ __forceinline__ uint4 assemble_light(const LightParams& lt, const float mu[3], const float wout[3],
                                                const float4& sh) {
  float wix = lt.pos[0] - mu[0], wiy = lt.pos[1] - mu[1], wiz = lt.pos[2] - mu[2];
  const float d = sqrtf(wix * wix + wiy * wiy + wiz * wiz);
  const float id = 1.f / d;
  wix *= id; wiy *= id; wiz *= id;
  // degree 0: the three degree-1 coefficients are zero
  float v = kY00 * sh.x + kY1 * (sh.y * wiy + sh.z * wiz + sh.w * wix);
  v = fminf(1.f, fmaxf(0.f, v));
  return make_uint4(pack2<F16>(wix, wiy), pack2<F16>(wiz, wout[0]), pack2<F16>(wout[1], wout[2]),
                    pack2<F16>(d, v));
}

// ---- TMEM helpers ---------------------------------------------------------------------------------
// The A operand of every layer lives in TMEM (tcgen05.mma with A from tensor memory): row m of the
// tile is TMEM lane m, and 32-bit column j of the operand holds the 16-bit pair (k = 2j, 2j + 1), low
// half first.  Only the weights are read from shared memory by the tensor core.
__device__ __forceinline__ void tmem_st4(uint32_t taddr, uint4 v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(v.x),
               "r"(v.y), "r"(v.z), "r"(v.w)
               : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t* w) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr),
               "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7])
               : "memory");
}
__device__ __forceinline__ void tmem_wait_st() {
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
// D[tmem] (+)= A[tmem] . B[smem desc]^T, kind::f16 (16-bit inputs, fp32 accumulate); ACC = false
// overwrites D.  The whole issuing warp executes this with warp-uniform operands; the instruction is
// predicated on `issue` (1 in one elected lane).
template <bool ACC>
__device__ __forceinline__ void umma_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t desc_b, uint32_t idesc,
                                        uint32_t issue) {
  asm volatile(
      "{\n\t.reg .pred p, q;\n\t"
      "setp.ne.u32 p, %4, 0;\n\t"
      "setp.ne.u32 q, %5, 0;\n\t"
      "@q tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(tmem_d), "r"(tmem_a), "l"(desc_b), "r"(idesc), "r"(ACC ? 1u : 0u), "r"(issue)
      : "memory");
}
// tcgen05.commit under the same predicate: arrives on the mbarrier when the MMAs issued so far complete
__device__ __forceinline__ void umma_commit_if(uint32_t bar, uint32_t issue) {
  asm volatile(
      "{\n\t.reg .pred q;\n\t"
      "setp.ne.u32 q, %1, 0;\n\t"
      "@q tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}"
      ::"r"(bar), "r"(issue)
      : "memory");
}
// 1 in one elected lane of the (converged) warp, 0 in the others
__device__ __forceinline__ uint32_t elect_one() {
  uint32_t e;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(e));
  return e;
}
// Makes this thread's A-operand writes visible to the tensor core before it signals a_ready.
__device__ __forceinline__ void a_publish() {
  tmem_wait_st();
  tc_fence_before();
}

// Writes the light-INDEPENDENT 16-byte chunks among [c_begin, c_end) of this thread's row of the layer-0
// A operand (chunk c = TMEM columns at0 + 4c .. 4c + 3 of this thread's lane): everything but chunk 1.
// The layer-0 operand has a TMEM region of its own, so this happens once per block of 128 Gaussians; per
// light only chunk 1 is rewritten (and the per-Gaussian feature is read from HBM / L2 once, not per light).
template <bool F16>
__device__ __forceinline__ void write_static(const MlpArgs& a, int64_t g, uint32_t at0, int c_begin,
                                             int c_end, const uint4* keep) {
#pragma unroll
  for (int c = 0; c < kKeepChunks; ++c)
    if (c != 1 && c >= c_begin && c < c_end) tmem_st4(at0 + 4 * c, keep[c]);
  const int F = a.plan.feat_dim;
  for (int c = max(c_begin, kKeepChunks); c < c_end; ++c) {
    const int j = (c - 5) * 8;
    float4 f0 = make_float4(0.f, 0.f, 0.f, 0.f), f1 = f0;
    if (j < F) f0 = *reinterpret_cast<const float4*>(a.feat + g * F + j);
    if (j + 4 < F) f1 = *reinterpret_cast<const float4*>(a.feat + g * F + j + 4);
    tmem_st4(at0 + 4 * c, make_uint4(pack2<F16>(f0.x, f0.y), pack2<F16>(f0.z, f0.w), pack2<F16>(f1.x, f1.y),
                                     pack2<F16>(f1.z, f1.w)));
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
// fine stamps inside the epilogue of thread 0 of CTA 0 (slot 0): code | clock, appended to slot 3's row
__device__ int g_fine_n;
#define TL_FINE(code)                                                               \
  do {                                                                              \
    if (blockIdx.x == 0 && threadIdx.x == 0 && g_fine_n < 500) g_timeline[3][g_fine_n++] = (clock64() << 4) | (code); \
  } while (0)
#else
#define TL_STAMP(code) do {} while (0)
#define TL_FINE(code) do {} while (0)
#endif

// ---- epilogue helpers --------------------------------------------------------------------------
// 16 accumulator columns of this thread's row, TMEM -> registers, asynchronously: the registers
// are valid only after tmem_wait_ld on the same array (which carries the data dependence).
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
template <int N>
__device__ __forceinline__ void tmem_wait_ld(uint32_t* r) {
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
  // empty volatile asms keep their order after the wait and make every later use of r[i] depend on it
#pragma unroll
  for (int i = 0; i < N; ++i) asm volatile("" : "+r"(r[i]));
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float* v) {
  uint32_t r[16];
  tmem_ld16_async(taddr, r);
  tmem_wait_ld<16>(r);
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
// 16-bit pair {lo, hi} = round-to-nearest-even of (max(lo, 0), max(hi, 0)): the ReLU rides on the convert
template <bool F16>
__device__ __forceinline__ uint32_t pack2_relu(float lo, float hi) {
  uint32_t d;
  if (F16) asm("cvt.rn.relu.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  else asm("cvt.rn.relu.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}

// activation + 16-bit convert of the 16 accumulator columns c0 .. c0 + 15 (bias already inside: it
// came through the tensor core) -> 8 columns of the next A operand, one tcgen05.st.
template <bool RELU, bool F16>
__device__ __forceinline__ void finish16(const uint32_t* r, uint32_t at, int c0, int activation, float slope) {
  uint32_t w[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const float lo = __uint_as_float(r[2 * i]), hi = __uint_as_float(r[2 * i + 1]);
    if (RELU) w[i] = pack2_relu<F16>(lo, hi);
    else w[i] = pack2<F16>(act_fn(lo, activation, slope), act_fn(hi, activation, slope));
  }
  tmem_st8(at + (uint32_t)(c0 >> 1), w);
}

// Hidden-stage epilogue of one thread: its share of the activated columns [0, n_act), in groups
// of 16, with the TMEM load of the next group in flight while the current one is finished (32-column
// loads were measured no faster and cost registers).  WPS = 4: all columns; WPS = 8: the two warps of a
// row quarter take alternate 32-column blocks.  d_taddr / at: this thread's lane base in the slot's
// accumulator / A operand.
template <int WPS_, bool RELU, bool F16>
__device__ __forceinline__ void hidden_epilogue(uint32_t d_taddr, uint32_t at, int n_act, int half,
                                                int activation, float slope) {
  constexpr int G = WPS_ == 4 ? 8 : 4;  // groups of 16 columns per thread for 128 columns
  uint32_t ra[16], rb[16];
  // group gi covers columns col(gi) .. +15
  auto col = [&](int gi) { return WPS_ == 4 ? 16 * gi : 32 * half + 64 * (gi >> 1) + 16 * (gi & 1); };
  if (col(0) + 16 <= n_act) tmem_ld16_async(d_taddr + col(0), ra);
#pragma unroll
  for (int gp = 0; gp < G / 2; ++gp) {
    const int c0 = col(2 * gp), c1 = col(2 * gp + 1);
    if (c0 + 16 > n_act) break;
    TL_FINE(8);
    tmem_wait_ld<16>(ra);
    TL_FINE(9);
    if (c1 + 16 <= n_act) tmem_ld16_async(d_taddr + c1, rb);
    finish16<RELU, F16>(ra, at, c0, activation, slope);
    TL_FINE(10);
    if (c1 + 16 > n_act) break;
    tmem_wait_ld<16>(rb);
    TL_FINE(11);
    if (2 * gp + 2 < G) {
      const int c2 = col(2 * gp + 2);
      if (c2 + 16 <= n_act) tmem_ld16_async(d_taddr + c2, ra);
    }
    finish16<RELU, F16>(rb, at, c1, activation, slope);
    TL_FINE(12);
  }
}

__device__ __forceinline__ float sigmoid_fast(float x) { return __fdividef(1.f, 1.f + __expf(-x)); }

constexpr int kMlpThreadsMax = 512;  // up to 16 warps: 4 slots x 4 warps or 2 slots x 8 warps

// Work distribution: a "unit" is a block of 128 Gaussians with all the lights of the batch; slot s of
// CTA b owns the units (i * slots + s) * gridDim.x + b, i = 0, 1, ...  Within a unit the lights are
// walked in order so that the light-independent inputs of a row are assembled once.
template <int WPS, bool RELU, bool F16>
__global__ void __launch_bounds__(kMlpThreadsMax, 1) mlp_kernel(const __grid_constant__ MlpArgs a) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  const MlpPlan& plan = a.plan;
  const int S = a.slots;
  uint8_t* sW = smem;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + plan.blob_bytes);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * kMaxSlots + 1);
  // bars[s] = a_ready of slot s, bars[kMaxSlots + s] = d_ready of slot s, bars[2 kMaxSlots] = weights landed

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

  // ---- prologue: barriers, weights to smem, TMEM, the constant-ones operand ----------------------
  // The packed weights (100-170 KB) come in with TMA bulk copies issued by one thread (32 KB each, completion
  // counted on an mbarrier): they land through the async proxy the tensor core reads with, and the other
  // threads go on to allocate TMEM and assemble their first rows meanwhile.  (Before: 16-byte LDG + STS by
  // every thread, ~20 round trips each, and a proxy fence.)
  const uint32_t bar_w = smem_u32(bars + 2 * kMaxSlots);
  if (tid == 0) {
    for (int s = 0; s < S; ++s) {
      mbar_init(smem_u32(bars + s), WPS * 32);
      mbar_init(smem_u32(bars + kMaxSlots + s), 1);
    }
    mbar_init(bar_w, 1);
    fence_barrier_init();
    if (a.plain_copy) mbar_arrive(bar_w);
    else mbar_expect_tx(bar_w, (uint32_t)plan.blob_bytes);
    // 4 KB pieces, every CTA starting at another one: all CTAs of the grid read the same blob at the same time,
    // and in the same order they would queue on the same L2 slices
    const int n_pieces = (plan.blob_bytes + 4095) / 4096;
    for (int q = 0; q < n_pieces && !a.plain_copy; ++q) {
      const int off = ((q + (int)blockIdx.x * 7) % n_pieces) * 4096;
      bulk_copy_g2s(smem_u32(sW + off), a.blob + off, (uint32_t)min(4096, plan.blob_bytes - off), bar_w);
    }
  }
  if (a.plain_copy) {  // measurement aid (SSSGS_MLP_PLAIN_COPY=1): the round-1 copy, 16-byte LDG + STS by every thread
    for (int i = tid * 16; i < plan.blob_bytes; i += blockDim.x * 16)
      *reinterpret_cast<uint4*>(sW + i) = *reinterpret_cast<const uint4*>(a.blob + i);
    fence_proxy_async();
  }
  if (warp == 0) tmem_alloc(smem_u32(tmem_slot), kTmemCols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const uint32_t ones_addr = tmem_base + (uint32_t)(kTmemCols - kOnesCols);
  if (warp < 4) {
    // A operand of the bias K step: k = 0, 1, 2 are 1.0 in every row (lane), k = 3 .. 15 are 0.
    // Warp w may only touch the TMEM lanes 32 w .. 32 w + 31.
    const uint32_t one = F16 ? 0x3C00u : 0x3F80u;
    const uint32_t w[8] = {one | (one << 16), one, 0u, 0u, 0u, 0u, 0u, 0u};
    tmem_st8(ones_addr + ((uint32_t)(warp * 32) << 16), w);
    tmem_wait_st();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();

  {
    // ===================== input assembly + epilogue warps =====================
    // a warp may only touch the TMEM lanes 32 * (warp % 4) .. +31: WPS is 4 or 8, so warp % 4 is
    // also the row quarter inside the slot
    const int slot = warp / WPS, wq = warp % WPS;
    const int quarter = wq & 3, half = wq >> 2;   // column half (WPS = 8)
    const int r = quarter * 32 + lane;            // row of the tile = TMEM lane
    // this thread's lane base in the slot's accumulator (taddr) and A operand (at)
    const uint32_t lane_base = tmem_base + ((uint32_t)(quarter * 32) << 16);
    const uint32_t taddr = lane_base + slot * a.d_stride;
    const uint32_t at = lane_base + a.a_base + slot * a.a_stride;
    const uint32_t at0 = lane_base + a.a0_base + slot * a.a0_stride;   // layer-0 operand
    const uint32_t th = lane_base + a.h_base + slot * 16;              // last stage's accumulator
    const uint32_t bar_a = smem_u32(bars + slot), bar_d = smem_u32(bars + kMaxSlots + slot);
    // The first warp of a slot also issues the slot's MMAs: once all rows of the A operand have
    // arrived (a_ready), it issues the bias step and the K steps of the stage and commits them to
    // d_ready.  A slot's pipeline is serial anyway (A operand -> MMA -> epilogue -> next A operand);
    // the tensor core is kept busy by the other slots.
    int tl_n = 0;
    (void)tl_n;
    uint32_t pa = 0;
    // warp-uniform copies of what the issue code needs (a shuffle from lane 0 tells the compiler so)
    const uint32_t issue = elect_one();
    const uint32_t u_d_addr = __shfl_sync(0xFFFFFFFFu, tmem_base + slot * a.d_stride, 0);
    const uint32_t u_h_addr = __shfl_sync(0xFFFFFFFFu, tmem_base + a.h_base + slot * 16, 0);
    const uint32_t u_a_addr = __shfl_sync(0xFFFFFFFFu, tmem_base + a.a_base + slot * a.a_stride, 0);
    const uint32_t u_a0_addr = __shfl_sync(0xFFFFFFFFu, tmem_base + a.a0_base + slot * a.a0_stride, 0);
    const uint32_t u_ones = __shfl_sync(0xFFFFFFFFu, ones_addr, 0);
    const uint32_t u_w_base = __shfl_sync(0xFFFFFFFFu, smem_u32(sW), 0);
    // FIRST / LAST are compile-time at every call site: with run-time selects of the operand addresses the
    // compiler moves them to vector registers and every MMA operand goes through R2UR again
    auto issue_stage = [&](int s_idx, auto first_tag, auto last_tag) {
      constexpr bool FIRST = decltype(first_tag)::value, LAST = decltype(last_tag)::value;
      if (wq != 0) return;
      TL_STAMP(0);
      mbar_wait(bar_a, pa);
      pa ^= 1u;
      tc_fence_after();
      TL_STAMP(1);
      {
        // the stage's fields are read with a run-time index: shuffled from lane 0 so that the compiler keeps
        // everything derived from them in uniform registers (no R2UR per MMA operand)
        const int st_n_pad = __shfl_sync(0xFFFFFFFFu, plan.st[s_idx].n_pad, 0);
        const int st_k_pad = __shfl_sync(0xFFFFFFFFu, plan.st[s_idx].k_pad, 0);
        const int st_w_off = __shfl_sync(0xFFFFFFFFu, plan.st[s_idx].w_off, 0);
        const uint32_t idesc = make_idesc(st_n_pad, F16);
        const uint32_t w_addr = u_w_base + (uint32_t)st_w_off;
        // stage 0 reads the layer-0 operand's own region; the last stage accumulates into its own 16 columns
        // (the next light's stage 0 may then be issued before the last stage's epilogue has read them)
        const uint32_t d_addr = LAST ? u_h_addr : u_d_addr;
        const uint32_t a_addr = FIRST ? u_a0_addr : u_a_addr;
        // bias step: ones . (hi, mid, lo)^T overwrites D; the stage's slot is the 16-column K step s % 4 of
        // bias block s / 4 (the descriptor's start address advances by 32 bytes per K step)
        const uint64_t dbias = make_desc(u_w_base + (uint32_t)(plan.bias_off + (s_idx >> 2) * plan.max_n * 128)) +
                               (uint64_t)((s_idx & 3) * 2);
        umma_ts<false>(d_addr, u_ones, dbias, idesc, issue);
        // one K step = 16 x 16 bit = 8 TMEM columns of A and 32 bytes inside a 128-byte swizzled row of
        // the weights; the second 64-wide K block starts n_pad * 128 bytes further
        const int ksteps = st_k_pad >> 4;
        const uint64_t db0 = make_desc(w_addr);
        const uint64_t db1 = make_desc(w_addr + st_n_pad * 128);
#pragma unroll
        for (int ks = 0; ks < 8; ++ks)
          if (ks < ksteps) umma_ts<true>(d_addr, a_addr + ks * 8, (ks < 4 ? db0 : db1) + (uint64_t)((ks & 3) * 2), idesc, issue);
        umma_commit_if(bar_d, issue);  // arrives when the MMAs above have completed
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
    if (wq == 0) mbar_wait(bar_w, 0);   // the issuing warps: the bulk copies of the weights have landed
    // The slots of a CTA should run out of phase (one slot's epilogue under the other's MMAs); started together
    // they tend to stay in step.  Slot s starts s * stagger clocks late (tuning aid SSSGS_MLP_STAGGER).
    if (slot > 0 && a.stagger > 0) {
      const long long t_go = clock64() + (long long)slot * a.stagger;
      while (clock64() < t_go) __nanosleep(100);
    }
    for (int64_t u = (int64_t)slot * gridDim.x + blockIdx.x; u < n_units; u += (int64_t)S * gridDim.x) {
      const int64_t row = (u / split) * kRows + r;
      const int light0 = (int)(u % split) * lights_per_unit;
      const int light1 = min(a.n_lights, light0 + lights_per_unit);
      const bool row_ok = row < n_rows;
      const int64_t row_c = row_ok ? row : n_rows - 1;
      const int64_t g = a.rows ? (int64_t)a.rows[row_c] : row_c;
      uint4 keep[kKeepChunks];
      float mu[3], wout[3];
      float4 sh = make_float4(0.f, 0.f, 0.f, 0.f);
      assemble_static<F16>(a, g, c_begin, c_end, keep, mu, wout, sh);
      // layer-0 operand of the block: light-independent chunks once, chunk 1 for the first light
      write_static<F16>(a, g, at0, c_begin, c_end, keep);
      if (c_begin == 0) tmem_st4(at0 + 4, assemble_light<F16>(a.lights.l[light0], mu, wout, sh));
      a_publish();
      mbar_arrive(bar_a);
      issue_stage(0, std::true_type{}, std::false_type{});
      for (int light = light0; light < light1; ++light) {
        float sss_keep[3] = {0.f, 0.f, 0.f};
        for (int s = 0; s < plan.n_stages; ++s) {
          const MlpStage& st = plan.st[s];
          mbar_wait(bar_d, pd);
          pd ^= 1u;
          tc_fence_after();
          TL_STAMP(3);
          // stage 0's MMAs have completed: the layer-0 operand is free for the next light's chunk 1 (published
          // with this stage's epilogue writes)
          if (s == 0 && light + 1 < light1 && c_begin == 0)
            tmem_st4(at0 + 4, assemble_light<F16>(a.lights.l[light + 1], mu, wout, sh));
          if (st.type == ST_HIDDEN || st.type == ST_HEAD_SPLIT_A) {
            // activated columns [0, n_act) -> 16 bit -> next stage's A operand
            hidden_epilogue<WPS, RELU, F16>(taddr, at, st.n_act, half, plan.activation, plan.leaky_slope);
            if (st.type == ST_HEAD_SPLIT_A && half == 0) {  // SSS logits sit right after the activated columns
              float v[16];
              tmem_ld16(taddr + st.n_act, v);
#pragma unroll
              for (int c = 0; c < 3; ++c) sss_keep[c] = sigmoid_fast(v[c]);
            }
            TL_STAMP(4);
            TL_FINE(13);
            a_publish();
            TL_FINE(14);
            mbar_arrive(bar_a);
            if (s + 1 == plan.n_stages - 1) issue_stage(s + 1, std::false_type{}, std::true_type{});
            else issue_stage(s + 1, std::false_type{}, std::false_type{});
          } else {
            // last stage: the next light's stage 0 goes to the tensor core first (its operand was published
            // with stage 0's epilogue, its accumulator is not the one read below), then the outputs
            if (light + 1 < light1) {
              tc_fence_before();
              mbar_arrive(bar_a);
              issue_stage(0, std::true_type{}, std::false_type{});
            }
            if (half == 0) {
              float v[16];
              tmem_ld16(th, v);
              float4 o;
              if (st.type == ST_HEAD_JOINT) {
                o.x = sigmoid_fast(v[0]);
                o.y = sigmoid_fast(v[1]);
                o.z = sigmoid_fast(v[2]);
                o.w = fmaxf(0.f, v[3]);
              } else {  // ST_HEAD_SPLIT_B
                o = make_float4(sss_keep[0], sss_keep[1], sss_keep[2], fmaxf(0.f, v[0]));
              }
              if (row_ok) {
                a.out_internal[(size_t)g * a.n_lights + light] = o;
                if (a.out_user)
                  *reinterpret_cast<float4*>(a.out_user + (int64_t)light * a.user_light_stride + g * 4) = o;
              }
            }
            TL_STAMP(5);
            tc_fence_before();  // TMEM reads are ordered before the next a_ready arrive
          }
        }
      }
    }
  }

  // ---- teardown ----------------------------------------------------------------------------------
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem_base, kTmemCols);
}

}  // namespace

// How a plan runs.  A slot (one 128-row tile in flight) owns, in TMEM: its fp32 accumulator (widest
// layer, rounded up to 32 columns), the 16-bit A operand of the hidden layers (widest input / 2
// columns), the layer-0 A operand (in_pad / 2 columns, written once per block of Gaussians) and the 16
// accumulator columns of the last stage; the last kOnesCols columns of the allocation hold the
// constant-ones operand of the bias steps.  At most 4 slots (16 warps).
struct MlpShape {
  int slots, wps, d_stride, h_base, a_base, a_stride, a0_base, a0_stride;
};
static MlpShape mlp_shape(const MlpPlan& plan) {
  const int d_cols = (plan.max_n + 31) / 32 * 32;
  const int a_cols = plan.max_k_bytes / (kRows * 128) * 32;  // K blocks of 64 x 16 bit = 32 columns each
  const int a0_cols = (plan.in_pad / 2 + 7) / 8 * 8;          // layer-0 operand (K steps of 8 columns)
  const int per_slot = d_cols + 16 + a_cols + a0_cols;
  MlpShape sh;
  sh.slots = (kTmemCols - kOnesCols) / per_slot;
  if (sh.slots > kMaxSlots) sh.slots = kMaxSlots;
  if (sh.slots < 1) sh.slots = 1;
  sh.wps = sh.slots <= 2 ? 8 : 4;
  {  // tuning aid: SSSGS_MLP_SHAPE=<slots><wps>, e.g. 24 = 2 slots, 4 warps per slot
    static int force = -1;
    if (force < 0) { const char* e = getenv("SSSGS_MLP_SHAPE"); force = e ? atoi(e) : 0; }
    if (force > 0) {
      const int slots = force / 10 % 10, wps = force % 10;
      if (slots >= 1 && slots <= sh.slots && (wps == 4 || wps == 8) && slots * wps <= 16) {
        sh.slots = slots; sh.wps = wps;
      }
    }
  }
  // all accumulators first (32-column granules), then the 16-column ones, then the operands
  sh.d_stride = d_cols;
  sh.h_base = sh.slots * d_cols;
  sh.a_base = sh.h_base + sh.slots * 16;
  sh.a_stride = a_cols;
  sh.a0_base = sh.a_base + sh.slots * a_cols;
  sh.a0_stride = a0_cols;
  return sh;
}

int mlp_smem_bytes(const MlpPlan& plan) {
  return plan.blob_bytes + (2 * kMaxSlots + 1) * 8 + 16 + 1024;
}

int launch_mlp_pack(const sssgs_mlp& mlp, const MlpPlan& plan, uint8_t* blob, cudaStream_t s) {
  launch_pdl(mlp_pack_kernel, dim3(32), dim3(256), 0, s, plan, mlp.params, mlp.dtype, blob);
  return 1;
}

int launch_mlp(const sssgs_gaussians& g, const MlpPlan& plan, const uint8_t* blob,
               const CamParams& cam, const LightBatch& lights, int n_lights,
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
  a.blob = blob;
  a.out_internal = out_internal; a.out_user = out_user; a.user_light_stride = user_light_stride;
  a.plan = plan;
  a.rows = rows; a.row_count = row_count; a.rows_out = rows_out;
  const MlpShape sh = mlp_shape(plan);
  a.slots = sh.slots; a.wps = sh.wps; a.d_stride = sh.d_stride; a.h_base = sh.h_base; a.a_base = sh.a_base;
  a.a_stride = sh.a_stride; a.a0_base = sh.a0_base; a.a0_stride = sh.a0_stride;
  {
    static int stagger = -1;
    if (stagger < 0) { const char* e = getenv("SSSGS_MLP_STAGGER"); stagger = e ? atoi(e) : 0; }
    a.stagger = stagger;
    static int plain = -1;
    if (plain < 0) { const char* e = getenv("SSSGS_MLP_PLAIN_COPY"); plain = e ? atoi(e) : 0; }
    a.plain_copy = plain;
  }
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
  const int v = (plan.f16 ? 4 : 0) + (a.wps == 8 ? 2 : 0) + (relu ? 1 : 0);
  switch (v) {
    case 0: return launch(mlp_kernel<4, false, false>);
    case 1: return launch(mlp_kernel<4, true, false>);
    case 2: return launch(mlp_kernel<8, false, false>);
    case 3: return launch(mlp_kernel<8, true, false>);
    case 4: return launch(mlp_kernel<4, false, true>);
    case 5: return launch(mlp_kernel<4, true, true>);
    case 6: return launch(mlp_kernel<8, false, true>);
    default: return launch(mlp_kernel<8, true, true>);
  }
}

}  // namespace sssgs

#ifdef SSSGS_MLP_TIMELINE
extern "C" int sssgs_debug_mlp_timeline(long long* out) {
  return (int)cudaMemcpyFromSymbol(out, sssgs::g_timeline, sizeof(long long) * sssgs::kMaxSlots * 512);
}
#endif

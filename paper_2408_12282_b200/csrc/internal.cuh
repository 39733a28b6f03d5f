// Internal declarations shared by the kernels of libsssgs (never installed; not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/sssgs.h"

#include <map>
#include <mutex>
#include <utility>

namespace sssgs {

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-DEVICE attribute of a kernel: the opt-in is
// remembered per (kernel, device ordinal of the calling thread's current device), so that contexts on
// several GPUs of one process each get it, and a warmed-up context makes no attribute call any more
// (CUDA-graph capture of sssgs_render).
inline cudaError_t ensure_dyn_smem(const void* kernel, int bytes) {
  static std::mutex mu;
  static std::map<std::pair<const void*, int>, int> done;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(mu);
  int& cur = done[std::make_pair(kernel, dev)];
  if (bytes > cur) {
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return e;
    cur = bytes;
  }
  return cudaSuccess;
}

// ---- programmatic dependent launch ------------------------------------------------------------
// The render path is a chain of short dependent kernels.  Each one is launched with the
// programmatic-stream-serialization attribute and starts with pdl_prologue(): it lets the NEXT
// kernel of the stream start launching once all of this kernel's CTAs are running, then waits
// until the PREVIOUS kernel has completed and flushed.  Launch latency and CTA start-up of a
// kernel thus overlap the tail of its predecessor; data dependences are unchanged (nothing is
// read or written before the wait).  Without the attribute both instructions are no-ops.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_prologue() {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
}
#endif
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem,
                              cudaStream_t s, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

// ---- constants of the method (S4) -----------------------------------
constexpr float kAlphaMin = 1.0f / 255.0f;
constexpr float kAlphaMax = 0.99f;
constexpr float kTMin = 1e-4f;
constexpr float kLowPass = 0.3f;
constexpr float kFrustumClamp = 1.3f;
constexpr float kDiscFloor = 0.1f;
constexpr float kRadiusSigma = 3.33f;
constexpr int kTile = SSSGS_TILE;

// ---- radix sort geometry --------------------------------------------------------------------
constexpr int kSortThreads = 256;
constexpr int kSortItemsMax = 15;
constexpr int kSortTileMax = kSortThreads * kSortItemsMax;  // keys per ticket, at most
constexpr uint32_t kSortFill = 148 * 4;                     // tickets that fill the machine
// keys per thread and ticket, by problem size: the smallest of {3, 7, 15} that needs no more
// than kSortFill tickets (15 beyond that)
__host__ __device__ inline int sort_items_for(uint32_t n) {
  if (n <= kSortFill * (uint32_t)kSortThreads * 3u) return 3;
  if (n <= kSortFill * (uint32_t)kSortThreads * 7u) return 7;
  return 15;
}
// rows of look-back status a pass over at most `cap` keys can need
__host__ __device__ inline uint32_t sort_status_rows(uint32_t cap) {
  const uint32_t per = (uint32_t)kSortThreads * (uint32_t)sort_items_for(cap);
  const uint32_t rows = (cap + per - 1) / per;
  return (cap > kSortFill * (uint32_t)kSortThreads * 3u && rows < kSortFill) ? kSortFill : rows;
}
constexpr int kRadixMax = 256;
constexpr int kLongListLog2 = 10;  // lists of >= 1024 entries are walked by more CTAs on small images
constexpr uint32_t kFlagAgg = 1u << 30;  // look-back status: aggregate of this tile only
constexpr uint32_t kFlagInc = 2u << 30;  // inclusive prefix up to and including this tile
constexpr uint32_t kFlagMask = 3u << 30;
constexpr uint32_t kValMask = ~kFlagMask;
constexpr int kSpinLimit = 1 << 24;  // bug trap for look-back waits (sets SSSGS_CNT_SORT_ERROR)

// Depth-sort passes whose digit is the same for all n keys are identity permutations and are
// skipped on the device (for an object in front of the camera the exponent byte of the depth
// usually is).  Counts the passes among [0, upto) that do run: a pass runs if its histogram has
// no bin holding all n keys; the last pass also runs if nothing ran before it, so that the
// sorted index array always exists.  Called by all 256 threads of a CTA; hist = 4 x 256 words.
#ifdef __CUDACC__
__device__ __forceinline__ int depth_passes_run(const uint32_t* __restrict__ hist, uint32_t n, int upto,
                                                bool* runs_last) {
  int ran = 0;
  bool r = true;
  for (int q = 0; q < upto; ++q) {
    const bool trivial = __syncthreads_or(hist[q * 256 + threadIdx.x] == n) != 0;
    r = !trivial || (q == 3 && ran == 0);
    ran += r ? 1 : 0;
  }
  if (runs_last) *runs_last = r;
  return ran;
}
#endif

// ---- emit (scan + expand) geometry ----------------------------------------------------------
constexpr int kEmitThreads = 256;
constexpr int kEmitChunk = kEmitThreads;  // Gaussians per ticket

struct CamParams {   // device copy of sssgs_camera plus derived values
  float R[9], t[3];
  float fx, fy, cx, cy, tanx, tany;
  int width, height;
  float znear;
  float bg[3];
  float pos[3];      // camera position in world space = -R^T t
  int tiles_x, tiles_y;
};

struct LightParams {
  float pos[3];
  float intensity[3];
};

constexpr int kMaxLightsPerPass = 8;
struct LightBatch {
  LightParams l[kMaxLightsPerPass];
};

// Device counters (uint32 each), zeroed once per camera.
enum {
  DC_NVIS = 0,
  DC_INSTANCES = 1,   // total I (unclamped)
  DC_OVERFLOW = 2,
  DC_SORT_ERROR = 3,
  DC_TICKET_BASE = 8, // tickets: one per ticketed kernel launch
  DC_RANGES_DONE = 24,   // blocks of ranges_kernel that have finished
  DC_CONTRIB_ROWS = 25,  // Gaussians kept by the visibility pre-pass (MLP rows of a sweep)
  DC_WC_CHUNKS = 26,     // weight cache: chunks handed out
  DC_WC_OVERFLOW = 27,   // weight cache: 1 if the pool ran out (the sweep then walks the lists again)
  DC_BWD_ROWS = 28,      // backward: rows of the light batch with a non-zero dL/d(mlp_out)
  DC_BWD_GOMAX = 29,     // backward: bits of the largest |dL/d(mlp_out)| of the light batch (follows DC_BWD_ROWS)
  DC_BVH_BOUNDS = 32,    // 6 words: box of the centres (sssgs_bake_visibility)
  DC_BUCKET_STARTS = 64, // 32 words: tiles with a list of at least 2^k entries, k = 0..31 (raster work order)
  DC_WORDS = 96
};

// Geometry buffers of one camera view.
struct GeomBuffers {
  float4* rec_a;      // [n] (pix_x, pix_y, depth, half2 support half-extents ex|ey)
  float4* rec_b;      // [n] (-log2e/2 conic a, -log2e conic b, -log2e/2 conic c, opacity)
  uint2* rect;        // [n] packed tile rect: x = x0 | x1<<16, y = y0 | y1<<16
  uint32_t* touched;  // [n]
  uint32_t* dkeys[2]; // [n] depth keys ping/pong
  uint32_t* dvals[2]; // [n] Gaussian index ping/pong
  uint32_t* ikeys[2]; // [cap] tile id of each instance ping/pong
  uint32_t* ivals[2]; // [cap] Gaussian index of each instance ping/pong
  uint2* ranges;      // [tiles]
  uint32_t* tile_order; // [tiles] tile ids, longest lists first (raster work order)
  uint32_t* tile_slot;  // [tiles + 1] scratch: lower bound of every tile id in the sorted instances
  uint32_t* hist;     // [6][256] digit histograms: 4 depth passes + 2 tile passes
  uint32_t* status;   // look-back status words, carved per pass
  uint32_t* counters; // [DC_WORDS]
};

// ---- weight cache of a light sweep ----------------------------------------------------------
// The compositing weights T_i alpha_i of a view do not depend on the light.  In a sweep the
// visibility pre-pass stores, per 8x4-pixel block (= warp) of every tile, the entries it blends
// -- (Gaussian id, depth) and the 32 per-pixel weights -- in chunks of 32 entries chained through
// `next`; the per-light walks then only stream those chunks and blend (no staging, culling, alpha
// evaluation or transmittance chain).  The pool is bounded: if it runs out, `overflow` is set and
// the sweep falls back to walking the lists.
constexpr int kWcChunk = 32;
struct WeightCache {
  uint32_t* head;     // [tiles * 8] first chunk of the block's chain
  uint32_t* count;    // [tiles * 8] entries in the chain
  uint32_t* next;     // [capacity] chunk -> next chunk
  uint2* hdr;         // [capacity * 32] (Gaussian id, bits(depth)) per entry
  float* weights;     // [capacity * 32 * 32] weight of the entry at each of the block's 32 pixels
  float* T;           // [H * W] final transmittance per pixel
  float4* gsum;       // [H * W * 3] sums of the light-independent channels (first light batch of the view)
  uint32_t* chunks;   // device counter: chunks handed out (DC_WC_CHUNKS)
  uint32_t* overflow; // device flag (DC_WC_OVERFLOW)
  uint32_t capacity;  // chunks in the pool
};

// ---- MLP description on the device ----------------------------------------------------------
constexpr int kMlpMaxStages = SSSGS_MAX_TRUNK + SSSGS_MAX_INC_HIDDEN + 1;
enum { ST_HIDDEN = 0, ST_HEAD_JOINT = 1, ST_HEAD_SPLIT_A = 2, ST_HEAD_SPLIT_B = 3 };
struct MlpStage {
  int k_pad;        // padded input width (multiple of 16)
  int n_pad;        // padded output width (multiple of 16)
  int n_act;        // outputs that go through the hidden activation and feed the next stage
  int type;
  int w_off;        // byte offset of this stage's packed bf16 weights in the blob
  // where the rows come from in the caller's packed parameter array (element offsets):
  // rows [0, src_rows[0]) from source 0, rows [src_rows[0], src_rows[0]+src_rows[1]) from source 1
  int src_w[2], src_b[2], src_rows[2];
  int src_k;        // un-padded input width (row length of the source matrices)
};
struct MlpPlan {
  int n_stages;
  int in_dim, in_pad;
  int feat_dim;
  int activation;
  float leaky_slope;
  int f16;          // tensor-core operand type: 1 = binary16 (default), 0 = bf16 (sssgs_mlp.compute)
  int blob_bytes;   // packed weights (all stages) + bias blocks, multiple of 1024
  int bias_off;     // byte offset of the bias blocks in the blob: block q = stages 4q .. 4q + 3, max_n x 128 bytes each
  int max_n;        // widest n_pad
  int max_k_bytes;  // bytes of the largest A tile (128 rows)
  MlpStage st[kMlpMaxStages];
};

// ---- launchers (each enqueues on `s`, returns the number of kernels launched) ---------------
int launch_pack_attr(const sssgs_gaussians& g, float4* attr, cudaStream_t s);
int launch_project(const sssgs_gaussians& g, const CamParams& cam, const GeomBuffers& gb, int tight,
                   cudaStream_t s);
int launch_sort_pass(const uint32_t* keys_in, const uint32_t* vals_in, uint32_t* keys_out,
                     uint32_t* vals_out, const uint32_t* count_ptr, uint32_t count_cap, int shift,
                     int bits, const uint32_t* hist, uint32_t* status, uint32_t* ticket,
                     uint32_t* err, int max_blocks, cudaStream_t s);
// depth pass `pass` of 4 over the ping-pong buffers keys[2] / vals[2] (skipped on the device when
// trivial, see depth_passes_run); hist4 = the 4 x 256 depth-digit histograms
int launch_depth_pass(uint32_t* const keys[2], uint32_t* const vals[2], uint32_t n, int pass,
                      const uint32_t* hist4, uint32_t* status, uint32_t* ticket, uint32_t* err,
                      int max_blocks, cudaStream_t s);
int launch_emit(int64_t n, const CamParams& cam, const GeomBuffers& gb, uint32_t cap, int tile_shift0, int tile_bits0, int tile_shift1, int tile_bits1,
                uint32_t* status, uint32_t* ticket, cudaStream_t s);
int launch_ranges(const uint32_t* sorted_tiles, const CamParams& cam, const GeomBuffers& gb,
                  uint32_t cap, uint2* ranges_user, int64_t* counters_out, int mlp_writes_rows,
                  cudaStream_t s);
int launch_export_lists(const uint32_t* sorted_tiles, const uint32_t* sorted_vals,
                        const GeomBuffers& gb, uint32_t cap, uint64_t* keys_out, uint32_t* vals_out,
                        cudaStream_t s);
int launch_mlp_pack(const sssgs_mlp& mlp, const MlpPlan& plan, uint8_t* blob, cudaStream_t s);
int launch_mlp(const sssgs_gaussians& g, const MlpPlan& plan, const uint8_t* blob,
               const CamParams& cam, const LightBatch& lights, int n_lights,
               float4* out_internal, float* out_user, int64_t user_light_stride, int max_ctas,
               const uint32_t* rows, const uint32_t* row_count, int64_t* rows_out, cudaStream_t s);
// "w/o deferred" variant (Tab. 2): Eq. 7 per Gaussian, then RGB compositing
int launch_shade_gaussians(int64_t n, int n_lights, const float* means, const float4* attr,
                           const CamParams& cam, const LightBatch& lights, float4* io, cudaStream_t s);
int launch_raster_forward(const CamParams& cam, int n_lights, const GeomBuffers& gb,
                          const uint32_t* sorted_vals, const float4* shaded, float* rgb,
                          int64_t frame_stride_px, cudaStream_t s);
// visibility pre-pass of a light sweep and its compaction
int launch_mark_contrib(const CamParams& cam, const GeomBuffers& gb, const uint32_t* sorted_vals,
                        uint8_t* contrib, const WeightCache* wc, cudaStream_t s);
// per-light walk over the weight cache (returns immediately on the device if the cache overflowed)
int launch_raster_cached(const CamParams& cam, const LightBatch& lights, int n_lights,
                         const GeomBuffers& gb, const WeightCache& wc, const float4* attr,
                         const float4* mlp_out, float* rgb, float* gbuf, float* aov_d, float* aov_s,
                         int64_t frame_stride_px, int sum_mode, int first_batch, cudaStream_t s);
int raster_reads_unblended_rows(int tiles);
// BVH of sssgs_bake_visibility (k_bvh.cu); nodes: internal 0 .. n-2 (root 0), leaf of sorted position k = n-1+k
struct BvhBuffers {
  uint32_t* code_of;       // [n] Morton code of Gaussian g
  uint32_t* sorted_codes;  // [n] codes in sorted order
  uint32_t* sorted_gid;    // [n] Gaussian index of sorted position k
  float4* leaf;            // [3n] (mu, o), (Sigma^-1 xx xy xz yy), (yz zz, cut-off, index)
  float4* box_lo;          // [2n-1] (min xyz, left child)
  float4* box_hi;          // [2n-1] (max xyz, right child)
  int* parent;             // [2n-1]
  uint32_t* flags;         // [n-1] refit arrival counters, zeroed by the caller
};
int launch_bvh_bounds(int64_t n, const float* means, uint32_t* bounds, int max_blocks, cudaStream_t s);
int launch_bvh_morton(int64_t n, const float* means, const uint32_t* bounds, uint32_t* keys, uint32_t* vals,
                      uint32_t* code_of, uint32_t* hist, int max_blocks, cudaStream_t s);
int launch_bvh_build(const sssgs_gaussians& g, const BvhBuffers& b, const uint32_t* depth_hist,
                     const uint32_t* vals0, const uint32_t* vals1, cudaStream_t s);
int launch_bvh_trace(int64_t n, const BvhBuffers& b, int n_dirs, const float* dirs, const float* weights, float t_min,
                     int n_coef, float* sh_out, float* vis_out, int positions, int num_sms, float4* scratch,
                     size_t scratch_bytes, cudaStream_t s);
int launch_compact_contrib(const uint8_t* contrib, int64_t n, uint32_t* rows, uint32_t* count,
                           int zero_rest, float4* out0, float4* out1, int lights, cudaStream_t s);
int launch_gather_precomputed(const float* pre, int64_t n, int n_lights, int64_t light_stride,
                              float4* out_internal, cudaStream_t s);
int launch_raster(const CamParams& cam, const LightBatch& lights, int n_lights,
                  const GeomBuffers& gb, const uint32_t* sorted_vals, const float4* attr,
                  const float4* mlp_out, float* rgb, float* gbuf, float* aov_d, float* aov_s,
                  int64_t frame_stride_px, int sum_mode, cudaStream_t s,
                  const uint32_t* only_if_set = nullptr);
// only_if_set: if given, the kernel returns at once unless *only_if_set != 0 (weight-cache fallback)
// sum_mode: 0 = one RGB frame per light; 1 = ONE frame = sum over the batch's lights + background
// term (first batch of a camera); 2 = add the batch's lights to the frame already there

// backward pass (k_backward.cu)
int launch_zero(float* p, int64_t n, cudaStream_t s);
int launch_project_backward(const sssgs_gaussians& g, const CamParams& cam, const float* g_mean2d, const float* g_conic,
                            const float* g_depth, float* d_means, float* d_scales, float* d_rot, cudaStream_t s);
int launch_shade_backward(const CamParams& cam, const LightBatch& lights, int n_lights, const float* gbuf,
                          const float* grad_rgb, const float* grad_gbuf_in, float* grad_gbuf, cudaStream_t s);
int launch_composite_backward(const CamParams& cam, int n_lights, const GeomBuffers& gb, const uint32_t* sorted_vals,
                              const float4* attr, const float4* mlp_out, int mlp_stride, const float* grad_gbuf,
                              float* g_opacity, float* g_mean2d, float* g_conic, float* g_depth, float* g_attr,
                              float* g_mlp_out, int64_t n, cudaStream_t s);
// row_count: two control words (rows listed, bits of max |dL/d(mlp_out)|); blob: kBwdBlobBytes, packed when `pack`
constexpr size_t kBwdBlobBytes = 4 * 32768 + 4096 + 5 * 512;
int launch_mlp_backward(const sssgs_gaussians& g, const sssgs_mlp& mlp, const CamParams& cam, const LightBatch& lights,
                        int n_lights, const float* g_mlp_out, float* g_params, uint32_t* row_list, uint32_t* row_count,
                        uint8_t* blob, bool pack, bool force_fp32, float* const input_grads[6], int num_sms, cudaStream_t s);

int mlp_smem_bytes(const MlpPlan& plan);

// reflectance-field relighting (k_relight.cu): out[p][c] = sum_l weights[l][c] frames[l][p][c]
int launch_relight(const float* frames, int n_light, int64_t n_pixels, const float* weights, float* out, int num_sms,
                   cudaStream_t s);

}  // namespace sssgs

// Tile binning (hot-path steps a4, a6): exclusive scan of tiles-touched in depth order fused
// with the expansion into (tile id, Gaussian) instances, the per-tile ranges, and the optional
// export of the sorted lists in the ABI's 64-bit key format.
//
// emit_kernel: persistent CTAs pull chunks of 256 depth-sorted Gaussians by ticket.  A chunk is
// scanned with warp shuffles, its global base comes from a decoupled look-back over the chunk
// totals (integer prefix sums: deterministic), and each warp expands its 32 Gaussians so that
// consecutive lanes write consecutive instances (a lane finds its Gaussian by a 5-step shuffle
// search over the warp's offsets), tile y then x ascending inside a Gaussian.  The CTA also
// accumulates the digit histograms of the tile ids for the tile sort.
// Traffic: 4+4+8 B read per Gaussian, 8 B written per instance.
#include "internal.cuh"

namespace sssgs {

namespace {

__device__ __forceinline__ uint32_t ld_volatile(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ void st_volatile(uint32_t* p, uint32_t v) {
  asm volatile("st.volatile.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

__global__ void __launch_bounds__(kEmitThreads)
emit_kernel(uint32_t n, const uint32_t* __restrict__ dvals0, const uint32_t* __restrict__ dvals1,
            const uint32_t* __restrict__ depth_hist, const uint32_t* __restrict__ touched, const uint2* __restrict__ rect, int tiles_x,
            uint32_t cap, uint32_t* __restrict__ ikeys, uint32_t* __restrict__ ivals,
            uint32_t* __restrict__ hist0, uint32_t* __restrict__ hist1, int shift0, int bits0,
            int shift1, int bits1, uint32_t* __restrict__ status, uint32_t* __restrict__ ticket,
            uint32_t* __restrict__ counters) {
  __shared__ uint32_t s_hist[2][kRadixMax];
  __shared__ uint32_t s_wsum[kEmitThreads / 32];
  __shared__ uint32_t s_ticket, s_base;

  const unsigned tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t nchunks = (n + kEmitChunk - 1) / kEmitChunk;
  const uint32_t mask0 = (1u << bits0) - 1u, mask1 = bits1 ? (1u << bits1) - 1u : 0u;
  pdl_prologue();
  s_hist[0][tid] = 0;
  s_hist[1][tid] = 0;
  // the depth-sorted index array sits in the buffer the last executed depth pass wrote
  const uint32_t* __restrict__ sorted_idx = (depth_passes_run(depth_hist, n, 4, nullptr) & 1) ? dvals1 : dvals0;

  while (true) {
    __syncthreads();
    if (tid == 0) s_ticket = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t t = s_ticket;
    if (t >= nchunks) break;

    // ---- one depth-sorted Gaussian per thread; scan of tiles-touched over the chunk -----------
    const uint32_t j = t * (uint32_t)kEmitChunk + tid;
    uint32_t g = 0, cnt = 0;
    uint2 r = make_uint2(0u, 0u);
    if (j < n) {
      g = sorted_idx[j];
      cnt = touched[g];
      r = rect[g];
    }
    uint32_t inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, inc, o);
      if (lane >= (unsigned)o) inc += v;
    }
    if (lane == 31) s_wsum[warp] = inc;
    __syncthreads();
    uint32_t wbase = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kEmitThreads / 32; ++w) {
      const uint32_t v = s_wsum[w];
      if ((unsigned)w < warp) wbase += v;
      total += v;
    }
    if (warp == 0) {
      // ---- decoupled look-back over chunk totals, one warp looking at 32 earlier chunks at a time --
      uint32_t excl = 0;
      if (t == 0) {
        if (lane == 0) st_volatile(status, kFlagInc | total);
      } else {
        if (lane == 0) st_volatile(status + t, kFlagAgg | total);
        int spins = 0;
        for (int64_t first = (int64_t)t - 1;;) {
          const int64_t idx = first - lane;
          const uint32_t v = idx >= 0 ? ld_volatile(status + idx) : kFlagInc;
          const unsigned inc = __ballot_sync(0xFFFFFFFFu, (v & kFlagMask) == kFlagInc);
          const unsigned none = __ballot_sync(0xFFFFFFFFu, (v & kFlagMask) == 0u);
          const int stop = inc ? __ffs(inc) - 1 : 31;            // nearest chunk with an inclusive prefix
          const unsigned need = stop == 31 ? 0xFFFFFFFFu : ((2u << stop) - 1u);
          if (none & need) {                                     // a chunk in between is not published yet
            if (++spins > kSpinLimit) {
              if (lane == 0) atomicExch(&counters[DC_SORT_ERROR], 2u);
              break;
            }
            __nanosleep(20);
            continue;
          }
          // a chunk total is at most 256 x 65536 = 2^24 and an inclusive prefix at most kValMask: the 32
          // values of a step sum to less than 2^32; the running prefix SATURATES at kValMask (2^30 - 1,
          // above any capacity) instead of wrapping, and saturation counts as overflow
          uint32_t val = lane <= stop ? (v & kValMask) : 0u;
#pragma unroll
          for (int o = 16; o >= 1; o >>= 1) val += __shfl_xor_sync(0xFFFFFFFFu, val, o);
          excl = (uint32_t)min((uint64_t)excl + val, (uint64_t)kValMask);
          if (inc) break;
          first -= 32;
        }
        if (lane == 0) st_volatile(status + t, kFlagInc | (uint32_t)min((uint64_t)excl + total, (uint64_t)kValMask));
      }
      if (lane == 0) {
        s_base = excl;
        if (t == nchunks - 1) {
          const uint32_t all = (uint32_t)min((uint64_t)excl + total, (uint64_t)kValMask);
          counters[DC_INSTANCES] = all;  // saturated at 2^30 - 1
          if (all > cap || all == kValMask) counters[DC_OVERFLOW] = 1u;
        }
      }
    }
    __syncthreads();

    // ---- expand, one warp per 32 Gaussians: consecutive lanes write consecutive instances ------
    const uint32_t woff = inc - cnt;                       // exclusive offset inside the warp
    const uint32_t wtotal = __shfl_sync(0xFFFFFFFFu, inc, 31);
    const uint32_t gbase = s_base + wbase;
    for (uint32_t ob = 0; ob < wtotal; ob += 32) {         // warp-uniform trip count
      const uint32_t o = ob + lane;
      // last lane l with woff[l] <= o (zero-count lanes share their successor's start)
      uint32_t lo = 0;
#pragma unroll
      for (int step = 16; step >= 1; step >>= 1) {
        const uint32_t cand = lo + step;
        const uint32_t v = __shfl_sync(0xFFFFFFFFu, woff, cand & 31);
        if (v <= o) lo = cand;
      }
      const uint32_t l_off = __shfl_sync(0xFFFFFFFFu, woff, lo);
      const uint32_t l_rx = __shfl_sync(0xFFFFFFFFu, r.x, lo);
      const uint32_t l_ry = __shfl_sync(0xFFFFFFFFu, r.y, lo);
      const uint32_t l_g = __shfl_sync(0xFFFFFFFFu, g, lo);
      const uint32_t dst = gbase + o;
      const bool ok = o < wtotal && dst < cap;
      if (ok) {
        const uint32_t k = o - l_off;
        const uint32_t x0 = l_rx & 0xFFFFu, x1 = l_rx >> 16, y0 = l_ry & 0xFFFFu;
        const uint32_t w = x1 - x0;
        // k < tiles touched <= 65536 and w <= 4096: the float quotient of (k + 0.5) / w floors exactly
        const uint32_t row = (uint32_t)__fdividef((float)k + 0.5f, (float)w);
        const uint32_t ty = y0 + row, tx = x0 + (k - row * w);
        const uint32_t tile = ty * (uint32_t)tiles_x + tx;
        ikeys[dst] = tile;
        ivals[dst] = l_g;
        // digit histograms of the tile id for the tile sort: the low digit differs between
        // neighbouring instances (x ascending), the high digit is mostly warp-uniform
        atomicAdd(&s_hist[0][(tile >> shift0) & mask0], 1u);
        if (bits1) {
          const uint32_t d1 = (tile >> shift1) & mask1;
          const unsigned act = __activemask();
          const uint32_t d1_first = __shfl_sync(act, d1, __ffs(act) - 1);
          if (__all_sync(act, d1 == d1_first)) {
            if (lane == (unsigned)(__ffs(act) - 1)) atomicAdd(&s_hist[1][d1], __popc(act));
          } else {
            atomicAdd(&s_hist[1][d1], 1u);
          }
        }
      }
    }
  }
  __syncthreads();
  if (s_hist[0][tid]) atomicAdd(&hist0[tid], s_hist[0][tid]);
  if (bits1 && s_hist[1][tid]) atomicAdd(&hist1[tid], s_hist[1][tid]);
}

// ranges[t] = [lower_bound(t), lower_bound(t+1)) over the sorted tile ids.  Every boundary i
// between two different neighbouring tile ids a < b defines lower_bound(t) = i for all t in
// (a, b] (the ends count as tile ids -1 and `tiles`), so one coalesced sweep over the sorted ids
// fills lb[0..tiles].  The last block to finish turns lb into ranges and builds the
// rasteriser's work order: tile ids bucketed by floor(log2(list length)) and laid out longest
// first, so that the longest lists start first and the tail of the raster kernel is short
// (order inside a bucket is arbitrary; it only schedules).
__global__ void __launch_bounds__(256)
ranges_kernel(const uint32_t* __restrict__ sorted_tiles, uint32_t* __restrict__ counters,
              uint32_t cap, int tiles, uint2* __restrict__ ranges, uint2* __restrict__ ranges_user,
              uint32_t* __restrict__ lb, uint32_t* __restrict__ tile_order,
              int64_t* __restrict__ counters_out, int mlp_writes_rows) {
  __shared__ uint32_t s_cnt[32], s_start[32];
  __shared__ bool s_last;
  pdl_prologue();
  const uint32_t n = min(counters[DC_INSTANCES], cap);
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i <= n; i += gridDim.x * 256u) {
    const int a = i == 0 ? -1 : (int)sorted_tiles[i - 1];
    const int b = i == n ? tiles : (int)sorted_tiles[i];
    for (int t = a + 1; t <= b; ++t) lb[t] = i;
  }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) s_last = atomicAdd(&counters[DC_RANGES_DONE], 1u) == gridDim.x - 1;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (threadIdx.x < 32) s_cnt[threadIdx.x] = 0;
  if (counters_out && threadIdx.x < SSSGS_NCOUNTERS) {
    int64_t v = 0;
    if (threadIdx.x == SSSGS_CNT_NVIS) v = counters[DC_NVIS];
    if (threadIdx.x == SSSGS_CNT_INSTANCES) v = counters[DC_INSTANCES];
    if (threadIdx.x == SSSGS_CNT_OVERFLOW) v = counters[DC_OVERFLOW];
    if (threadIdx.x == SSSGS_CNT_SORT_ERROR) v = counters[DC_SORT_ERROR];
    // SSSGS_CNT_MLP_ROWS is written by the MLP kernel (possibly before this kernel runs)
    if (threadIdx.x != SSSGS_CNT_MLP_ROWS || !mlp_writes_rows) counters_out[threadIdx.x] = v;
  }
  __syncthreads();
  for (int t = threadIdx.x; t < tiles; t += 256) {
    const uint32_t b0 = __ldcg(&lb[t]), b1 = __ldcg(&lb[t + 1]);
    ranges[t] = make_uint2(b0, b1);
    if (ranges_user) ranges_user[t] = make_uint2(b0, b1);
    atomicAdd(&s_cnt[32u - __clz(b1 - b0)], 1u);  // bucket 0: empty list, else floor(log2(len)) + 1
  }
  __syncthreads();
  if (threadIdx.x < 32) {
    uint32_t start = 0;
    for (int k = 31; k > (int)threadIdx.x; --k) start += s_cnt[k];
    s_start[threadIdx.x] = start;
    // bucket b holds lengths in [2^(b-1), 2^b): `start` tiles have at least 2^b entries, and come first
    counters[DC_BUCKET_STARTS + threadIdx.x] = start;
  }
  __syncthreads();
  for (int t = threadIdx.x; t < tiles; t += 256) {
    const uint32_t len = __ldcg(&lb[t + 1]) - __ldcg(&lb[t]);
    tile_order[atomicAdd(&s_start[32u - __clz(len)], 1u)] = (uint32_t)t;
  }
}

// Optional export in the ABI format: key = tile << 32 | bits(depth), value = Gaussian index.
__global__ void __launch_bounds__(256)
export_lists_kernel(const uint32_t* __restrict__ sorted_tiles, const uint32_t* __restrict__ sorted_vals,
                    const float4* __restrict__ rec_a, const uint32_t* __restrict__ counters,
                    uint32_t cap, uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out) {
  pdl_prologue();
  const uint32_t n = min(counters[DC_INSTANCES], cap);
  for (uint32_t j = blockIdx.x * 256u + threadIdx.x; j < n; j += gridDim.x * 256u) {
    const uint32_t g = sorted_vals[j];
    if (keys_out) keys_out[j] = ((uint64_t)sorted_tiles[j] << 32) | __float_as_uint(rec_a[g].z);
    if (vals_out) vals_out[j] = g;
  }
}

// Compaction of the visibility pre-pass: indices of the Gaussians with contrib[g] != 0, in
// blocks (order inside a block ascending; blocks in arrival order -- the order only decides which
// MLP tile a row lands in, never a result).  With zero_rest, the MLP-output rows of the other
// Gaussians are zero-filled in both output buffers (see raster_reads_unblended_rows).
__global__ void __launch_bounds__(256)
compact_contrib_kernel(const uint8_t* __restrict__ contrib, uint32_t n, uint32_t* __restrict__ rows,
                       uint32_t* __restrict__ count, int zero_rest, float4* __restrict__ out0,
                       float4* __restrict__ out1, int lights) {
  __shared__ uint32_t s_w[8], s_base;
  pdl_prologue();
  const uint32_t g = blockIdx.x * 256u + threadIdx.x;
  const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool on = g < n && contrib[g] != 0;
  const unsigned m = __ballot_sync(0xFFFFFFFFu, on);
  if (lane == 0) s_w[warp] = __popc(m);
  __syncthreads();
  uint32_t before = 0, total = 0;
#pragma unroll
  for (int w = 0; w < 8; ++w) {
    if ((unsigned)w < warp) before += s_w[w];
    total += s_w[w];
  }
  if (threadIdx.x == 0) s_base = total ? atomicAdd(count, total) : 0u;
  __syncthreads();
  if (on) rows[s_base + before + __popc(m & ((1u << lane) - 1u))] = g;
  if (zero_rest && g < n && !on) {
    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int l = 0; l < lights; ++l) {
      out0[(size_t)g * lights + l] = z;
      out1[(size_t)g * lights + l] = z;
    }
  }
}

}  // namespace

int launch_compact_contrib(const uint8_t* contrib, int64_t n, uint32_t* rows, uint32_t* count,
                           int zero_rest, float4* out0, float4* out1, int lights, cudaStream_t s) {
  if (n == 0) return 0;
  launch_pdl(compact_contrib_kernel, dim3((unsigned)((n + 255) / 256)), dim3(256), 0, s, contrib, (uint32_t)n,
             rows, count, zero_rest, out0, out1, lights);
  return 1;
}

int launch_emit(int64_t n, const CamParams& cam, const GeomBuffers& gb, uint32_t cap, int tile_shift0, int tile_bits0, int tile_shift1, int tile_bits1,
                uint32_t* status, uint32_t* ticket, cudaStream_t s) {
  if (n == 0) return 0;
  int64_t blocks = (n + kEmitChunk - 1) / kEmitChunk;
  if (blocks > 148 * 8) blocks = 148 * 8;  // 8 CTAs fit an SM: a chunk is a chain of dependent loads
  launch_pdl(emit_kernel, dim3((unsigned)blocks), dim3(kEmitThreads), 0, s,
      (uint32_t)n, gb.dvals[0], gb.dvals[1], gb.hist, gb.touched, gb.rect, cam.tiles_x, cap, gb.ikeys[0], gb.ivals[0],
      gb.hist + 4 * 256, gb.hist + 5 * 256, tile_shift0, tile_bits0, tile_shift1, tile_bits1, status,
      ticket, gb.counters);
  return 1;
}

int launch_ranges(const uint32_t* sorted_tiles, const CamParams& cam, const GeomBuffers& gb,
                  uint32_t cap, uint2* ranges_user, int64_t* counters_out, int mlp_writes_rows,
                  cudaStream_t s) {
  const int tiles = cam.tiles_x * cam.tiles_y;
  int64_t blocks = ((int64_t)cap + 1 + 1023) / 1024;
  if (blocks > 148 * 8) blocks = 148 * 8;
  launch_pdl(ranges_kernel, dim3((unsigned)blocks), dim3(256), 0, s, sorted_tiles, gb.counters, cap, tiles, gb.ranges,
                                                 ranges_user, gb.tile_slot, gb.tile_order, counters_out, mlp_writes_rows);
  return 1;
}

int launch_export_lists(const uint32_t* sorted_tiles, const uint32_t* sorted_vals,
                        const GeomBuffers& gb, uint32_t cap, uint64_t* keys_out, uint32_t* vals_out,
                        cudaStream_t s) {
  int64_t blocks = ((int64_t)cap + 255) / 256;
  if (blocks > 148 * 8) blocks = 148 * 8;
  if (blocks < 1) blocks = 1;
  launch_pdl(export_lists_kernel, dim3((unsigned)blocks), dim3(256), 0, s, sorted_tiles, sorted_vals, gb.rec_a,
                                                       gb.counters, cap, keys_out, vals_out);
  return 1;
}

}  // namespace sssgs

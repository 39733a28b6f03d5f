// Tile binning (hot-path steps a4, a6): exclusive scan of tiles-touched in depth order fused
// with the expansion into (tile id, Gaussian) instances, the per-tile ranges, and the optional
// export of the sorted lists in the ABI's 64-bit key format.
//
// emit_kernel: persistent CTAs pull chunks of 1024 depth-sorted Gaussians by ticket.  A chunk
// is scanned in shared memory, its global base comes from a decoupled look-back over the
// chunk totals (integer prefix sums: deterministic), and the instances are written by
// consecutive threads to consecutive addresses (each thread finds its Gaussian by binary
// search in the chunk's offsets), tile y then x ascending inside a Gaussian.  The CTA also
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
emit_kernel(uint32_t n, const uint32_t* __restrict__ sorted_idx,
            const uint32_t* __restrict__ touched, const uint2* __restrict__ rect, int tiles_x,
            uint32_t cap, uint32_t* __restrict__ ikeys, uint32_t* __restrict__ ivals,
            uint32_t* __restrict__ hist0, uint32_t* __restrict__ hist1, int shift0, int bits0,
            int shift1, int bits1, uint32_t* __restrict__ status, uint32_t* __restrict__ ticket,
            uint32_t* __restrict__ counters) {
  __shared__ uint32_t s_off[kEmitChunk + 1];
  __shared__ uint32_t s_g[kEmitChunk];
  __shared__ uint2 s_rect[kEmitChunk];
  __shared__ uint32_t s_hist[2][kRadixMax];
  __shared__ uint32_t s_wsum[kEmitThreads / 32];
  __shared__ uint32_t s_ticket, s_base;

  const unsigned tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t nchunks = (n + kEmitChunk - 1) / kEmitChunk;
  const uint32_t mask0 = (1u << bits0) - 1u, mask1 = bits1 ? (1u << bits1) - 1u : 0u;
  s_hist[0][tid] = 0;
  s_hist[1][tid] = 0;

  while (true) {
    __syncthreads();
    if (tid == 0) s_ticket = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t t = s_ticket;
    if (t >= nchunks) break;

    // ---- load 4 consecutive sorted positions per thread, scan tiles-touched -----------------
    uint32_t c[kEmitItems], sum = 0;
#pragma unroll
    for (int k = 0; k < kEmitItems; ++k) {
      const uint32_t j = t * (uint32_t)kEmitChunk + tid * kEmitItems + k;
      uint32_t g = 0, cnt = 0;
      uint2 r = make_uint2(0u, 0u);
      if (j < n) {
        g = sorted_idx[j];
        cnt = touched[g];
        r = rect[g];
      }
      s_g[tid * kEmitItems + k] = g;
      s_rect[tid * kEmitItems + k] = r;
      c[k] = cnt;
      sum += cnt;
    }
    uint32_t inc = sum;
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
    uint32_t run = wbase + inc - sum;
#pragma unroll
    for (int k = 0; k < kEmitItems; ++k) {
      s_off[tid * kEmitItems + k] = run;
      run += c[k];
    }
    if (tid == 0) {
      s_off[kEmitChunk] = total;
      // ---- decoupled look-back over chunk totals ------------------------------------------
      uint32_t excl = 0;
      if (t == 0) {
        st_volatile(status, kFlagInc | total);
      } else {
        st_volatile(status + t, kFlagAgg | total);
        int spins = 0;
        for (uint32_t tt = t; tt-- > 0;) {
          uint32_t v = ld_volatile(status + tt);
          while ((v & kFlagMask) == 0u) {
            if (++spins > kSpinLimit) {
              atomicExch(&counters[DC_SORT_ERROR], 2u);
              v = kFlagInc;
              break;
            }
            __nanosleep(32);
            v = ld_volatile(status + tt);
          }
          excl += v & kValMask;
          if (v & kFlagInc) break;
        }
        st_volatile(status + t, kFlagInc | ((excl + total) & kValMask));
      }
      s_base = excl;
      if (t == nchunks - 1) {
        const uint32_t all = excl + total;
        counters[DC_INSTANCES] = all;
        if (all > cap) counters[DC_OVERFLOW] = 1u;
      }
    }
    __syncthreads();
    const uint32_t base = s_base;

    // ---- expand: consecutive threads write consecutive instances ----------------------------
    for (uint32_t ob = 0; ob < total; ob += kEmitThreads) {  // warp-uniform trip count
      const uint32_t o = ob + tid;
      bool ok = false;
      uint32_t tile = 0;
      if (o < total) {
        // last e with s_off[e] <= o  (zero-count entries share their successor's start)
        uint32_t lo = 0, hi = kEmitChunk;  // invariant: s_off[lo] <= o < s_off[hi]
        while (hi - lo > 1) {
          const uint32_t mid = (lo + hi) >> 1;
          if (s_off[mid] <= o) lo = mid; else hi = mid;
        }
        const uint32_t k = o - s_off[lo];
        const uint2 r = s_rect[lo];
        const uint32_t x0 = r.x & 0xFFFFu, x1 = r.x >> 16, y0 = r.y & 0xFFFFu;
        const uint32_t w = x1 - x0;
        const uint32_t ty = y0 + k / w, tx = x0 + k % w;
        tile = ty * (uint32_t)tiles_x + tx;
        const uint32_t dst = base + o;
        ok = dst < cap;
        if (ok) {
          ikeys[dst] = tile;
          ivals[dst] = s_g[lo];
        }
      }
      // warp-aggregated digit histograms
      const unsigned act = __ballot_sync(0xFFFFFFFFu, ok);
      if (ok) {
        const uint32_t d0 = (tile >> shift0) & mask0;
        unsigned peers = __match_any_sync(act, d0);
        if ((peers & ((1u << lane) - 1u)) == 0) atomicAdd(&s_hist[0][d0], __popc(peers));
        if (bits1) {
          const uint32_t d1 = (tile >> shift1) & mask1;
          peers = __match_any_sync(act, d1);
          if ((peers & ((1u << lane) - 1u)) == 0) atomicAdd(&s_hist[1][d1], __popc(peers));
        }
      }
    }
  }
  __syncthreads();
  if (s_hist[0][tid]) atomicAdd(&hist0[tid], s_hist[0][tid]);
  if (bits1 && s_hist[1][tid]) atomicAdd(&hist1[tid], s_hist[1][tid]);
}

// ranges[t] = [lower_bound(t), lower_bound(t+1)) over the sorted tile ids (one thread per tile).
// The last block to finish also builds the rasteriser's work order: tile ids bucketed by
// floor(log2(list length)) and laid out longest first, so that the longest lists start first and
// the tail of the raster kernel is short (order inside a bucket is arbitrary; it only schedules).
__global__ void __launch_bounds__(256)
ranges_kernel(const uint32_t* __restrict__ sorted_tiles, uint32_t* __restrict__ counters,
              uint32_t cap, int tiles, uint2* __restrict__ ranges, uint2* __restrict__ ranges_user,
              uint32_t* __restrict__ tile_slot, uint32_t* __restrict__ tile_order) {
  __shared__ uint32_t s_start[32];
  __shared__ bool s_last;
  const int t = blockIdx.x * 256 + threadIdx.x;
  if (t < tiles) {
    const uint32_t n = min(counters[DC_INSTANCES], cap);
    uint32_t res[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const uint32_t target = (uint32_t)t + q;
      uint32_t lo = 0, hi = n;  // first index with key >= target
      while (lo < hi) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        if (sorted_tiles[mid] < target) lo = mid + 1; else hi = mid;
      }
      res[q] = lo;
    }
    ranges[t] = make_uint2(res[0], res[1]);
    if (ranges_user) ranges_user[t] = make_uint2(res[0], res[1]);
    const uint32_t len = res[1] - res[0];
    const uint32_t bucket = 32u - __clz(len);  // 0 for empty lists, else floor(log2(len)) + 1
    const uint32_t rank = atomicAdd(&counters[DC_BUCKET_BASE + bucket], 1u);
    tile_slot[t] = (bucket << 20) | rank;
  }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) s_last = atomicAdd(&counters[DC_RANGES_DONE], 1u) == gridDim.x - 1;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (threadIdx.x < 32) {
    uint32_t start = 0;
    for (int b = 31; b > (int)threadIdx.x; --b) start += atomicAdd(&counters[DC_BUCKET_BASE + b], 0u);
    s_start[threadIdx.x] = start;
  }
  __syncthreads();
  for (int u = threadIdx.x; u < tiles; u += 256) {
    const uint32_t slot = __ldcg(&tile_slot[u]);
    tile_order[s_start[slot >> 20] + (slot & 0xFFFFFu)] = (uint32_t)u;
  }
}

// Optional export in the ABI format: key = tile << 32 | bits(depth), value = Gaussian index.
__global__ void __launch_bounds__(256)
export_lists_kernel(const uint32_t* __restrict__ sorted_tiles, const uint32_t* __restrict__ sorted_vals,
                    const float4* __restrict__ rec_a, const uint32_t* __restrict__ counters,
                    uint32_t cap, uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out,
                    int64_t* __restrict__ counters_out) {
  const uint32_t n = min(counters[DC_INSTANCES], cap);
  if (counters_out && blockIdx.x == 0 && threadIdx.x < SSSGS_NCOUNTERS) {
    int64_t v = 0;
    if (threadIdx.x == SSSGS_CNT_NVIS) v = counters[DC_NVIS];
    if (threadIdx.x == SSSGS_CNT_INSTANCES) v = counters[DC_INSTANCES];
    if (threadIdx.x == SSSGS_CNT_OVERFLOW) v = counters[DC_OVERFLOW];
    if (threadIdx.x == SSSGS_CNT_SORT_ERROR) v = counters[DC_SORT_ERROR];
    counters_out[threadIdx.x] = v;
  }
  for (uint32_t j = blockIdx.x * 256u + threadIdx.x; j < n; j += gridDim.x * 256u) {
    const uint32_t g = sorted_vals[j];
    if (keys_out) keys_out[j] = ((uint64_t)sorted_tiles[j] << 32) | __float_as_uint(rec_a[g].z);
    if (vals_out) vals_out[j] = g;
  }
}

}  // namespace

int launch_emit(int64_t n, const CamParams& cam, const GeomBuffers& gb, const uint32_t* sorted_idx,
                uint32_t cap, int tile_shift0, int tile_bits0, int tile_shift1, int tile_bits1,
                uint32_t* status, uint32_t* ticket, cudaStream_t s) {
  if (n == 0) return 0;
  int64_t blocks = (n + kEmitChunk - 1) / kEmitChunk;
  if (blocks > 148 * 4) blocks = 148 * 4;
  emit_kernel<<<(unsigned)blocks, kEmitThreads, 0, s>>>(
      (uint32_t)n, sorted_idx, gb.touched, gb.rect, cam.tiles_x, cap, gb.ikeys[0], gb.ivals[0],
      gb.hist + 4 * 256, gb.hist + 5 * 256, tile_shift0, tile_bits0, tile_shift1, tile_bits1, status,
      ticket, gb.counters);
  return 1;
}

int launch_ranges(const uint32_t* sorted_tiles, const CamParams& cam, const GeomBuffers& gb,
                  uint32_t cap, uint2* ranges_user, cudaStream_t s) {
  const int tiles = cam.tiles_x * cam.tiles_y;
  ranges_kernel<<<(tiles + 255) / 256, 256, 0, s>>>(sorted_tiles, gb.counters, cap, tiles, gb.ranges,
                                                    ranges_user, gb.tile_slot, gb.tile_order);
  return 1;
}

int launch_export_lists(const uint32_t* sorted_tiles, const uint32_t* sorted_vals,
                        const GeomBuffers& gb, uint32_t cap, uint64_t* keys_out, uint32_t* vals_out,
                        int64_t* counters_out, cudaStream_t s) {
  int64_t blocks = ((int64_t)cap + 255) / 256;
  if (blocks > 148 * 8) blocks = 148 * 8;
  if (blocks < 1) blocks = 1;
  if (!keys_out && !vals_out) blocks = 1;
  export_lists_kernel<<<(unsigned)blocks, 256, 0, s>>>(sorted_tiles, sorted_vals, gb.rec_a,
                                                       gb.counters, cap, keys_out, vals_out,
                                                       counters_out);
  return 1;
}

}  // namespace sssgs

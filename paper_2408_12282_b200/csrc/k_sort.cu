// One-sweep LSD radix sort pass (hot-path step a5), hand-written: no CUB/Thrust.
//
// The tile lists of the method ("efficiently designed splatting technique", L68
// "layered sequenced Gaussians") are, per tile, the overlapping Gaussians ordered by
// (depth, index).  We obtain exactly that order with two stable LSD radix sorts
// (DESIGN.md "Sort"): (1) all Gaussians by the 32 bits of their depth, (2) the expanded
// (tile, Gaussian) instances -- emitted in depth order -- by tile id only.  Both use this
// kernel: one pass = one digit of <= 8 bits of a 32-bit key with a 32-bit payload.
//
// Structure of a pass (persistent CTAs pulling tickets, so a CTA only ever waits on tickets
// that are already running -> forward progress):
//   1. load 256 x 15 keys warp-striped (coalesced), rank them per warp with __match_any_sync
//      (stable: item order, then lane order), combine the per-warp digit counts,
//   2. publish the CTA's digit counts and resolve its global offsets by decoupled look-back
//      over the status words of earlier tickets (flag and 30-bit count share one word, so no
//      fence is needed),
//   3. reorder keys/payloads through shared memory into digit order and write each digit run
//      to its global position with consecutive threads writing consecutive addresses.
// HBM traffic per pass: 8 B read + 8 B written per element (4 B written on a payload-only
// final pass); the digit histograms come from the producing kernels (project / emit).
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

// exclusive scan of one value per thread over a 256-thread CTA; tmp = 8 words of smem.
__device__ __forceinline__ uint32_t block_excl_scan_256(uint32_t v, uint32_t* tmp) {
  const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
    if (lane >= (unsigned)o) inc += t;
  }
  if (lane == 31) tmp[warp] = inc;
  __syncthreads();
  uint32_t wbase = 0;
#pragma unroll
  for (int w = 0; w < 8; ++w)
    if ((unsigned)w < warp) wbase += tmp[w];
  __syncthreads();
  return wbase + inc - v;
}

__global__ void __launch_bounds__(kSortThreads)
radix_pass_kernel(const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                  uint32_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out,
                  const uint32_t* __restrict__ count_ptr, uint32_t count_cap, int shift, int bits,
                  const uint32_t* __restrict__ hist, uint32_t* __restrict__ status,
                  uint32_t* __restrict__ ticket, uint32_t* __restrict__ err) {
  __shared__ uint32_t s_keys[kSortTile];
  __shared__ uint32_t s_vals[kSortTile];
  __shared__ uint32_t s_wcnt[kSortThreads / 32][kRadixMax];
  __shared__ uint32_t s_binstart[kRadixMax];
  __shared__ uint32_t s_digstart[kRadixMax];
  __shared__ uint32_t s_gbase[kRadixMax];
  __shared__ uint32_t s_tmp[8];
  __shared__ uint32_t s_ticket;

  const unsigned tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t n = count_ptr ? min(*count_ptr, count_cap) : count_cap;
  const uint32_t ntiles = (n + kSortTile - 1) / kSortTile;
  const uint32_t radix = 1u << bits, mask = radix - 1u;

  // start of every digit bin in the output = exclusive scan of the global histogram
  {
    const uint32_t h = tid < radix ? hist[tid] : 0u;
    const uint32_t ex = block_excl_scan_256(h, s_tmp);
    s_binstart[tid] = ex;
  }

  while (true) {
    __syncthreads();  // also protects s_keys/s_vals/s_wcnt of the previous ticket
    if (tid == 0) s_ticket = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t t = s_ticket;
    if (t >= ntiles) break;

    // ---- 1. load + per-warp stable ranking ------------------------------------------------
    const uint32_t tile_base = t * (uint32_t)kSortTile;
    const uint32_t tile_count = min((uint32_t)kSortTile, n - tile_base);
    uint32_t key[kSortItems], val[kSortItems];
    uint32_t rank[kSortItems];
    const uint32_t first = tile_base + warp * (32u * kSortItems) + lane;
#pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
      const uint32_t idx = first + 32u * i;
      const bool ok = idx < n;
      key[i] = ok ? keys_in[idx] : 0xFFFFFFFFu;
      val[i] = ok ? (vals_in ? vals_in[idx] : idx) : 0u;
    }
    for (uint32_t d = lane; d < radix; d += 32) s_wcnt[warp][d] = 0;
    __syncwarp();
#pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
      const uint32_t d = (key[i] >> shift) & mask;
      const unsigned peers = __match_any_sync(0xFFFFFFFFu, d);
      const uint32_t r = __popc(peers & ((1u << lane) - 1u));
      const uint32_t base = s_wcnt[warp][d];
      __syncwarp();
      if (r == 0) s_wcnt[warp][d] = base + __popc(peers);
      __syncwarp();
      rank[i] = base + r;
    }
    __syncthreads();

    // ---- combine warps: per digit exclusive prefix over warps, CTA total -------------------
    uint32_t total = 0;
    if (tid < radix) {
#pragma unroll
      for (int w = 0; w < kSortThreads / 32; ++w) {
        const uint32_t c = s_wcnt[w][tid];
        s_wcnt[w][tid] = total;
        total += c;
      }
      // padding keys (0xFFFFFFFF, only in the last ticket) were ranked last in the last bin
      if (tid == mask) total -= (uint32_t)kSortTile - tile_count;
    }
    const uint32_t dig_start = block_excl_scan_256(total, s_tmp);
    if (tid < radix) s_digstart[tid] = dig_start;

    // ---- 2. decoupled look-back --------------------------------------------------------------
    if (tid < radix) {
      uint32_t* my = status + (size_t)t * kRadixMax + tid;
      uint32_t excl = 0;
      if (t == 0) {
        st_volatile(my, kFlagInc | total);
      } else {
        st_volatile(my, kFlagAgg | total);
        int spins = 0;
        for (uint32_t tt = t; tt-- > 0;) {
          const uint32_t* p = status + (size_t)tt * kRadixMax + tid;
          uint32_t v = ld_volatile(p);
          while ((v & kFlagMask) == 0u) {
            if (++spins > kSpinLimit) {
              atomicExch(err, 1u);
              v = kFlagInc;  // give up: result undefined, but no hang
              break;
            }
            __nanosleep(32);
            v = ld_volatile(p);
          }
          excl += v & kValMask;
          if (v & kFlagInc) break;
        }
        st_volatile(my, kFlagInc | ((excl + total) & kValMask));
      }
      s_gbase[tid] = s_binstart[tid] + excl - dig_start;
    }
    __syncthreads();

    // ---- 3. reorder through shared memory, then coalesced scatter ----------------------------
#pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
      const uint32_t d = (key[i] >> shift) & mask;
      const uint32_t pos = s_digstart[d] + s_wcnt[warp][d] + rank[i];
      s_keys[pos] = key[i];
      s_vals[pos] = val[i];
    }
    __syncthreads();
    for (uint32_t j = tid; j < tile_count; j += kSortThreads) {
      const uint32_t k = s_keys[j];
      const uint32_t dst = s_gbase[(k >> shift) & mask] + j;
      if (keys_out) keys_out[dst] = k;
      vals_out[dst] = s_vals[j];
    }
  }
}

}  // namespace

int launch_sort_pass(const uint32_t* keys_in, const uint32_t* vals_in, uint32_t* keys_out,
                     uint32_t* vals_out, const uint32_t* count_ptr, uint32_t count_cap, int shift,
                     int bits, const uint32_t* hist, uint32_t* status, uint32_t* ticket,
                     uint32_t* err, int max_blocks, cudaStream_t s) {
  if (count_cap == 0) return 0;
  int64_t blocks = ((int64_t)count_cap + kSortTile - 1) / kSortTile;
  if (blocks > max_blocks) blocks = max_blocks;
  radix_pass_kernel<<<(unsigned)blocks, kSortThreads, 0, s>>>(
      keys_in, vals_in, keys_out, vals_out, count_ptr, count_cap, shift, bits, hist, status, ticket,
      err);
  return 1;
}

}  // namespace sssgs

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
//   1. load 256 x ITEMS keys (ITEMS = 3, 7 or 15 by problem size) warp-striped (coalesced), rank them per warp (lanes with the same digit, found with one ballot per digit bit)
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

constexpr int kLookW = 8;  // look-back status words in flight per thread

struct SortSmem {
  uint32_t keys[kSortTileMax];
  uint32_t vals[kSortTileMax];
  uint32_t wcnt[kSortThreads / 32][kRadixMax];
  uint32_t binstart[kRadixMax];
  uint32_t digstart[kRadixMax];
  uint32_t gbase[kRadixMax];
  uint32_t tmp[8];
  uint32_t ticket;
};

// Lanes of the warp whose digit equals this lane's: one ballot per digit bit (measured faster than
// __match_any_sync on sm_100: 3 M keys x 4 passes 0.144 -> 0.109 ms).
__device__ __forceinline__ unsigned same_digit_lanes(uint32_t d, uint32_t mask) {
  unsigned pe = 0xFFFFFFFFu;
  for (uint32_t b = 1; b <= mask; b <<= 1) {
    const unsigned bal = __ballot_sync(0xFFFFFFFFu, (d & b) != 0u);
    pe &= (d & b) ? bal : ~bal;
  }
  return pe;
}

// Processes tickets of 256 x ITEMS keys until the ticket counter runs out.
template <int ITEMS>
__device__ __forceinline__ void sort_tickets(SortSmem& sm, const uint32_t* __restrict__ keys_in,
                                             const uint32_t* __restrict__ vals_in,
                                             uint32_t* __restrict__ keys_out,
                                             uint32_t* __restrict__ vals_out, uint32_t n, int shift,
                                             uint32_t radix, uint32_t mask,
                                             uint32_t* __restrict__ status,
                                             uint32_t* __restrict__ ticket, uint32_t* __restrict__ err) {
  constexpr uint32_t TILE = kSortThreads * ITEMS;
  const unsigned tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t ntiles = (n + TILE - 1) / TILE;
  // the first ticket was drawn at kernel entry (its latency overlaps the histogram scan)
  for (bool first_ticket = true;; first_ticket = false) {
    __syncthreads();  // also protects keys/vals/wcnt of the previous ticket
    if (!first_ticket) {
      if (ntiles <= gridDim.x) break;  // one ticket per CTA covers everything
      if (tid == 0) sm.ticket = atomicAdd(ticket, 1u);
      __syncthreads();
    }
    const uint32_t t = sm.ticket;
    if (t >= ntiles) break;

    // ---- 1. load + per-warp stable ranking ------------------------------------------------
    const uint32_t tile_base = t * TILE;
    const uint32_t tile_count = min(TILE, n - tile_base);
    uint32_t key[ITEMS], rank[ITEMS];
    unsigned peers[ITEMS];
    const uint32_t first = tile_base + warp * (32u * ITEMS) + lane;
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
      const uint32_t idx = first + 32u * i;
      const bool ok = idx < n;
      key[i] = ok ? keys_in[idx] : 0xFFFFFFFFu;
    }
    for (uint32_t d = lane; d < radix; d += 32) sm.wcnt[warp][d] = 0;
    // Short tickets (latency-bound small sorts): the matches of all items are independent of each
    // other and are issued back to back.  Long tickets keep the match inside the loop: 15 more live
    // registers would cost a resident CTA per SM, and large sorts are bandwidth-bound.
    constexpr bool kHoist = ITEMS <= 7;
    if (kHoist) {
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) peers[i] = same_digit_lanes((key[i] >> shift) & mask, mask);
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
      const uint32_t d = (key[i] >> shift) & mask;
      const unsigned pe = kHoist ? peers[i] : same_digit_lanes(d, mask);
      const uint32_t r = __popc(pe & ((1u << lane) - 1u));
      const uint32_t base = sm.wcnt[warp][d];
      __syncwarp();
      if (r == 0) sm.wcnt[warp][d] = base + __popc(pe);
      __syncwarp();
      rank[i] = base + r;
    }
    __syncthreads();

    // ---- combine warps: per digit exclusive prefix over warps, CTA total -------------------
    uint32_t total = 0;
    if (tid < radix) {
#pragma unroll
      for (int w = 0; w < kSortThreads / 32; ++w) {
        const uint32_t c = sm.wcnt[w][tid];
        sm.wcnt[w][tid] = total;
        total += c;
      }
      // padding keys (0xFFFFFFFF, only in the last ticket) were ranked last in the last bin
      if (tid == mask) total -= TILE - tile_count;
    }
    const uint32_t dig_start = block_excl_scan_256(total, sm.tmp);
    if (tid < radix) sm.digstart[tid] = dig_start;

    // ---- 2. decoupled look-back --------------------------------------------------------------
    if (tid < radix) {
      uint32_t* my = status + (size_t)t * kRadixMax + tid;
      uint32_t excl = 0;
      if (t == 0) {
        st_volatile(my, kFlagInc | total);
      } else {
        st_volatile(my, kFlagAgg | total);
        // walk back over earlier tickets, kLookW status words in flight at a time (the loads are
        // independent; only a word that is not published yet is re-read)
        int spins = 0;
        bool found = false;
        for (int64_t tt = (int64_t)t - 1; !found; tt -= kLookW) {
          uint32_t v[kLookW];
#pragma unroll
          for (int k = 0; k < kLookW; ++k)
            v[k] = tt - k >= 0 ? ld_volatile(status + (size_t)(tt - k) * kRadixMax + tid) : kFlagInc;
#pragma unroll
          for (int k = 0; k < kLookW; ++k) {
            if (!found) {
              while ((v[k] & kFlagMask) == 0u) {
                if (++spins > kSpinLimit) {
                  atomicExch(err, 1u);
                  v[k] = kFlagInc;  // give up: result undefined, but no hang
                  break;
                }
                __nanosleep(20);
                v[k] = ld_volatile(status + (size_t)(tt - k) * kRadixMax + tid);
              }
              excl += v[k] & kValMask;
              found = (v[k] & kFlagInc) != 0u;
            }
          }
        }
        st_volatile(my, kFlagInc | ((excl + total) & kValMask));
      }
      sm.gbase[tid] = sm.binstart[tid] + excl - dig_start;
    }
    __syncthreads();

    // ---- 3. reorder through shared memory, then coalesced scatter ----------------------------
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
      const uint32_t d = (key[i] >> shift) & mask;
      const uint32_t pos = sm.digstart[d] + sm.wcnt[warp][d] + rank[i];
      sm.keys[pos] = key[i];
      // the payload is only read here (fewer live registers while ranking): L2 serves it
      const uint32_t idx = first + 32u * i;
      sm.vals[pos] = idx < n ? (vals_in ? vals_in[idx] : idx) : 0u;
    }
    __syncthreads();
    for (uint32_t j = tid; j < tile_count; j += kSortThreads) {
      const uint32_t k = sm.keys[j];
      const uint32_t dst = sm.gbase[(k >> shift) & mask] + j;
      if (keys_out) keys_out[dst] = k;
      vals_out[dst] = sm.vals[j];
    }
  }
}

// depth_pass >= 0: pass `depth_pass` of the 4-pass depth sort over the ping-pong buffers
// (k0,v0) <-> (k1,v1); `hist` then points at all four histograms and trivial passes are skipped.
// depth_pass < 0: a plain pass from (k0,v0) to (k1,v1) with its own histogram.
__global__ void __launch_bounds__(kSortThreads, 4)
radix_pass_kernel(uint32_t* __restrict__ k0, uint32_t* __restrict__ v0, uint32_t* __restrict__ k1,
                  uint32_t* __restrict__ v1, const uint32_t* __restrict__ count_ptr,
                  uint32_t count_cap, int shift, int bits, const uint32_t* __restrict__ hist,
                  uint32_t* __restrict__ status, uint32_t* __restrict__ ticket,
                  uint32_t* __restrict__ err, int depth_pass) {
  __shared__ SortSmem sm;
  const unsigned tid = threadIdx.x;
  pdl_prologue();
  if (tid == 0) sm.ticket = atomicAdd(ticket, 1u);
  const uint32_t n = count_ptr ? min(*count_ptr, count_cap) : count_cap;
  const uint32_t radix = 1u << bits, mask = radix - 1u;
  const uint32_t *keys_in = k0, *vals_in = v0;
  uint32_t *keys_out = k1, *vals_out = v1;
  if (depth_pass >= 0) {
    bool runs;
    const int ran = depth_passes_run(hist, n, depth_pass + 1, &runs);
    if (!runs) return;
    const int before = ran - 1;  // passes that ran before this one
    if (before & 1) { keys_in = k1; vals_in = v1; keys_out = k0; vals_out = v0; }
    if (before == 0) vals_in = nullptr;      // nothing permuted yet: payload = index
    if (depth_pass == 3) keys_out = nullptr; // the keys are not needed after the last pass
    hist += depth_pass * 256;
  }

  // start of every digit bin in the output = exclusive scan of the global histogram
  {
    const uint32_t h = tid < radix ? hist[tid] : 0u;
    const uint32_t ex = block_excl_scan_256(h, sm.tmp);
    sm.binstart[tid] = ex;
  }
  // ticket size by problem size (uniform over the grid): small inputs are split finely so that
  // every SM gets work, large ones use long tickets that amortise the look-back
  const int items = sort_items_for(n);
  if (items == 3)
    sort_tickets<3>(sm, keys_in, vals_in, keys_out, vals_out, n, shift, radix, mask, status, ticket, err);
  else if (items == 7)
    sort_tickets<7>(sm, keys_in, vals_in, keys_out, vals_out, n, shift, radix, mask, status, ticket, err);
  else
    sort_tickets<15>(sm, keys_in, vals_in, keys_out, vals_out, n, shift, radix, mask, status, ticket, err);
}

}  // namespace

int launch_sort_pass(const uint32_t* keys_in, const uint32_t* vals_in, uint32_t* keys_out,
                     uint32_t* vals_out, const uint32_t* count_ptr, uint32_t count_cap, int shift,
                     int bits, const uint32_t* hist, uint32_t* status, uint32_t* ticket,
                     uint32_t* err, int max_blocks, cudaStream_t s) {
  if (count_cap == 0) return 0;
  int64_t blocks = (int64_t)sort_status_rows(count_cap);
  if (blocks > max_blocks) blocks = max_blocks;
  launch_pdl(radix_pass_kernel, dim3((unsigned)blocks), dim3(kSortThreads), 0, s,
             const_cast<uint32_t*>(keys_in), const_cast<uint32_t*>(vals_in), keys_out, vals_out, count_ptr,
             count_cap, shift, bits, hist, status, ticket, err, -1);
  return 1;
}

int launch_depth_pass(uint32_t* const keys[2], uint32_t* const vals[2], uint32_t n, int pass,
                      const uint32_t* hist4, uint32_t* status, uint32_t* ticket, uint32_t* err,
                      int max_blocks, cudaStream_t s) {
  if (n == 0) return 0;
  int64_t blocks = (int64_t)sort_status_rows(n);
  if (blocks > max_blocks) blocks = max_blocks;
  launch_pdl(radix_pass_kernel, dim3((unsigned)blocks), dim3(kSortThreads), 0, s, keys[0], vals[0], keys[1],
             vals[1], (const uint32_t*)nullptr, n, 8 * pass, 8, hist4, status, ticket, err, pass);
  return 1;
}

}  // namespace sssgs

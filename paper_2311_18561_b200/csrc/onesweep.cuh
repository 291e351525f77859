// onesweep.cuh -- stage a3: stable LSD radix sort of (u64 key, u32 value) pairs, one
// HBM read + one HBM write of the payload per digit pass ("onesweep": the per-tile
// digit offsets are resolved with a decoupled look-back chained across tiles inside
// the scatter kernel instead of a separate upsweep/scan/downsweep per pass).
// Implements PAPER.md:L70 ("Sorting the Gaussians according to their depth") on the
// (tile | depth) keys of DESIGN.md S11; ties keep their input order (stable).
#pragma once

#include "common.cuh"

namespace pvg {

constexpr int OS_RADIX_BITS = 8;
constexpr int OS_RADIX = 1 << OS_RADIX_BITS;
constexpr int OS_MAX_PASSES = 8;

struct SortPlan {
  int num_passes;
  int shift[OS_MAX_PASSES];
  int bits[OS_MAX_PASSES];
};

// Split [begin_bit, end_bit) into ceil(B/8) passes of near-equal width (14 -> 7+7).
inline SortPlan make_sort_plan(int begin_bit, int end_bit) {
  SortPlan p{};
  const int B = end_bit - begin_bit;
  p.num_passes = (B + OS_RADIX_BITS - 1) / OS_RADIX_BITS;
  int at = begin_bit;
  for (int i = 0; i < p.num_passes; ++i) {
    const int left = end_bit - at, passes_left = p.num_passes - i;
    const int b = (left + passes_left - 1) / passes_left;
    p.shift[i] = at;
    p.bits[i] = b;
    at += b;
  }
  return p;
}

// Lanes of the warp holding the same digit as the caller. One vote.ballot per digit bit:
// on sm_100a MATCH.ANY runs on the address-divergence unit at ~64 cycles per warp
// instruction per SM and caps a sort pass near 40% of HBM bandwidth (profiles/), while
// ballots issue on the regular pipes. `bits` is warp-uniform.
__device__ __forceinline__ uint32_t digit_peers(uint32_t d, int bits) {
  uint32_t peers = 0xffffffffu;
#pragma unroll
  for (int b = 0; b < OS_RADIX_BITS; ++b) {
    if (b < bits) {
      const bool one = (d >> b) & 1u;
      const uint32_t m = __ballot_sync(0xffffffffu, one);
      peers &= one ? m : ~m;
    }
  }
  return peers;
}

// ---- digit histograms of every pass in one read of the keys ---------------------------
constexpr int HIST_THREADS = 512;
constexpr int HIST_ITEMS = 8;

__global__ void __launch_bounds__(HIST_THREADS)
onesweep_histogram_kernel(const uint64_t* __restrict__ keys, uint64_t n, const __grid_constant__ SortPlan plan,
                          uint32_t* __restrict__ hist /* [passes][256] */) {
  __shared__ uint32_t s_hist[OS_MAX_PASSES * OS_RADIX];
  for (int k = threadIdx.x; k < plan.num_passes * OS_RADIX; k += HIST_THREADS) s_hist[k] = 0;
  __syncthreads();
  // block-uniform trip count; equal digits inside a warp are aggregated before the atomic
  // (tile-id digits of neighbouring instances are nearly always equal)
  constexpr uint64_t CH = (uint64_t)HIST_THREADS * HIST_ITEMS;
  const uint32_t lt = lanemask_lt();
  for (uint64_t base = (uint64_t)blockIdx.x * CH; base < n; base += (uint64_t)gridDim.x * CH) {
    uint64_t k[HIST_ITEMS];
#pragma unroll
    for (int u = 0; u < HIST_ITEMS; ++u) {
      const uint64_t idx = base + (uint64_t)u * HIST_THREADS + threadIdx.x;
      k[u] = idx < n ? __ldcs(keys + idx) : 0;
    }
#pragma unroll
    for (int u = 0; u < HIST_ITEMS; ++u) {
      const bool ok = base + (uint64_t)u * HIST_THREADS + threadIdx.x < n;
      for (int p = 0; p < plan.num_passes; ++p) {
        const uint32_t d = (uint32_t)(k[u] >> plan.shift[p]) & ((1u << plan.bits[p]) - 1u);
        const uint32_t live = __ballot_sync(0xffffffffu, ok);
        const uint32_t peers = digit_peers(d, plan.bits[p]) & live;
        if (ok && (peers & lt) == 0) atomicAdd(&s_hist[p * OS_RADIX + d], (uint32_t)__popc(peers));
      }
    }
  }
  __syncthreads();
  for (int k = threadIdx.x; k < plan.num_passes * OS_RADIX; k += HIST_THREADS) {
    const uint32_t v = s_hist[k];
    if (v) atomicAdd(&hist[k], v);
  }
}

// exclusive scan of each pass's 256-bin histogram (one block per pass, 256 threads)
__global__ void __launch_bounds__(OS_RADIX)
onesweep_scan_hist_kernel(uint32_t* __restrict__ hist) {
  __shared__ uint32_t s_warp[OS_RADIX / 32];
  uint32_t* h = hist + blockIdx.x * OS_RADIX;
  const uint32_t v = h[threadIdx.x];
  uint32_t incl = v;
  const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= d) incl += t;
  }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  uint32_t wex = 0;
  for (uint32_t w = 0; w < warp; ++w) wex += s_warp[w];
  h[threadIdx.x] = wex + incl - v;
}

// ---- one digit pass -------------------------------------------------------------------
template <int THREADS, int ITEMS>
struct OnesweepSmem {
  static constexpr int WARPS = THREADS / 32;
  static constexpr int TILE = THREADS * ITEMS;
  uint64_t keys[TILE];
  uint32_t vals[TILE];
  uint32_t warp_hist[WARPS * OS_RADIX];  // per-warp digit counts, then per-warp exclusive offsets
  uint32_t bin_start[OS_RADIX];          // tile-local start of each digit in sorted order
  uint32_t out_base[OS_RADIX];           // global index of the digit's first key MINUS bin_start
  uint32_t warp_sums[OS_RADIX / 32];
  uint32_t tile;
};

// Keys of a tile are read warp-striped (warp w owns ITEMS*32 consecutive keys, lane l its
// elements l, l+32, ...), ranked inside the warp with ballots (stable: earlier rounds and
// lower lanes come first), combined across warps per digit, resolved against earlier
// tiles by look-back, re-ordered through shared memory and written out in digit runs so
// that stores are coalesced.
template <int THREADS, int ITEMS>
__global__ void __launch_bounds__(THREADS, 2)
onesweep_pass_kernel(const uint64_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                     uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out, uint64_t n,
                     int shift, int bits, const uint32_t* __restrict__ hist_excl /* [256] this pass */,
                     uint64_t* __restrict__ lookback /* [tiles][256], zeroed */,
                     uint32_t* __restrict__ ticket /* zeroed */) {
  using Smem = OnesweepSmem<THREADS, ITEMS>;
  constexpr int WARPS = Smem::WARPS;
  constexpr int TILE = Smem::TILE;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem& s = *reinterpret_cast<Smem*>(smem_raw);

  const uint32_t tid = threadIdx.x, lane = lane_id(), warp = tid >> 5;
  if (tid == 0) s.tile = atomicAdd(ticket, 1u);
  for (int k = tid; k < WARPS * OS_RADIX; k += THREADS) s.warp_hist[k] = 0;
  __syncthreads();
  const uint32_t tile = s.tile;
  const uint64_t tile_base = (uint64_t)tile * TILE;
  const uint32_t tile_n = (uint32_t)min((uint64_t)TILE, n - tile_base);
  const uint32_t mask = (1u << bits) - 1u;

  // 1. load (warp-striped); padding keys are all-ones: they rank after every real key of
  //    the last digit and are never written
  const uint32_t wbase = warp * (ITEMS * 32) + lane;
  uint64_t key[ITEMS];
  uint32_t val[ITEMS];
#pragma unroll
  for (int j = 0; j < ITEMS; ++j) {
    const uint32_t li = wbase + j * 32;
    key[j] = li < tile_n ? __ldcs(keys_in + tile_base + li) : ~0ull;
  }
#pragma unroll
  for (int j = 0; j < ITEMS; ++j) {
    const uint32_t li = wbase + j * 32;
    val[j] = li < tile_n ? __ldcs(vals_in + tile_base + li) : 0u;
  }

  // 2. rank inside the warp
  uint32_t* wh = s.warp_hist + warp * OS_RADIX;
  uint16_t rank[ITEMS];
  const uint32_t lt = lanemask_lt();
#pragma unroll
  for (int j = 0; j < ITEMS; ++j) {
    const uint32_t d = (uint32_t)(key[j] >> shift) & mask;
    const uint32_t peers = digit_peers(d, bits);
    const uint32_t before = wh[d];
    __syncwarp();
    if ((peers & lt) == 0) wh[d] = before + __popc(peers);
    __syncwarp();
    rank[j] = (uint16_t)(before + __popc(peers & lt));
  }
  __syncthreads();

  // 3. per digit: exclusive scan of the warp counts over warps -> tile count
  uint32_t tile_count = 0;
  if (tid < OS_RADIX) {
#pragma unroll
    for (int w = 0; w < WARPS; ++w) {
      const uint32_t c = s.warp_hist[w * OS_RADIX + tid];
      s.warp_hist[w * OS_RADIX + tid] = tile_count;
      tile_count += c;
    }
    // 4. publish the tile's digit count, then resolve the exclusive prefix over earlier tiles
    uint64_t* my = lookback + (uint64_t)tile * OS_RADIX + tid;
    uint64_t excl = 0;
    if (tile == 0) {
      st_relaxed_u64(my, LB_FLAG_PREFIX | tile_count);
    } else {
      st_relaxed_u64(my, LB_FLAG_AGG | tile_count);
      int64_t p = (int64_t)tile - 1;
      while (true) {
        const uint64_t v = ld_relaxed_u64(lookback + (uint64_t)p * OS_RADIX + tid);
        const uint64_t flag = v & LB_FLAG_MASK;
        if (flag == 0) continue;  // that tile holds an earlier ticket: it is running
        excl += v & LB_VALUE_MASK;
        if (flag == LB_FLAG_PREFIX) break;
        --p;
      }
      st_relaxed_u64(my, LB_FLAG_PREFIX | (excl + tile_count));
    }
    // 5. exclusive scan of the tile counts over digits -> local bin starts
    uint32_t incl = tile_count;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
      if (lane >= d) incl += t;
    }
    if (lane == 31) s.warp_sums[warp] = incl;
    // warps 0..7 hold the digits; they meet at a named barrier of 256 threads
    asm volatile("bar.sync 1, %0;" ::"n"(OS_RADIX));
    uint32_t wex = 0;
    for (uint32_t w = 0; w < warp; ++w) wex += s.warp_sums[w];
    const uint32_t start = wex + incl - tile_count;
    s.bin_start[tid] = start;
    s.out_base[tid] = hist_excl[tid] + (uint32_t)excl - start;  // mod 2^32; n < 2^32
  }
  __syncthreads();

  // 6. scatter into shared memory in sorted order
#pragma unroll
  for (int j = 0; j < ITEMS; ++j) {
    const uint32_t d = (uint32_t)(key[j] >> shift) & mask;
    const uint32_t p = s.bin_start[d] + wh[d] + rank[j];
    s.keys[p] = key[j];
    s.vals[p] = val[j];
  }
  __syncthreads();

  // 7. coalesced write-out of digit runs (real keys occupy local positions [0, tile_n))
  for (uint32_t p = tid; p < tile_n; p += THREADS) {
    const uint64_t k = s.keys[p];
    const uint32_t d = (uint32_t)(k >> shift) & mask;
    const uint32_t o = s.out_base[d] + p;
    keys_out[o] = k;
    vals_out[o] = s.vals[p];
  }
}

}  // namespace pvg

// scan_dup.cuh -- stage a2, first half: exclusive prefix scan, in visiting order, of the number
// of items each Gaussian emits -- its tile count, or the number of 8x8-tile blocks its rectangle
// touches (blockbin.cuh). PAPER.md:L61 tile-based rasterisation; S11.
#pragma once

#include "common.cuh"

namespace pvg {

#ifndef PVG_SCAN_THREADS
#define PVG_SCAN_THREADS 512
#define PVG_SCAN_ITEMS 8
#endif
constexpr int SCAN_THREADS = PVG_SCAN_THREADS;
constexpr int SCAN_ITEMS = PVG_SCAN_ITEMS;   // a multiple of 4 (128-bit loads and stores)
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

// blocks of 8 x 8 tiles touched by the rectangle packed in the upper half of a sorted depth key
// (x0, y0, x1, y1, 8 bits each; preprocess.cuh); culled Gaussians carry depth bits 0xFFFFFFFF
__device__ __forceinline__ uint32_t scan_block_count(uint64_t key) {
  if ((uint32_t)key == 0xFFFFFFFFu) return 0u;
  const uint32_t r = (uint32_t)(key >> 32);
  const uint32_t x0 = r & 0xFFu, y0 = (r >> 8) & 0xFFu, x1 = (r >> 16) & 0xFFu, y1 = r >> 24;
  return ((x1 >> 3) - (x0 >> 3) + 1u) * ((y1 >> 3) - (y0 >> 3) + 1u);
}

// Single-pass chained scan with decoupled look-back. Warp-aggregated: per-thread
// serial sums -> warp shuffles -> one partial per warp -> block aggregate, which is
// published in a 64-bit status word (flag | value) and resolved against predecessor
// tiles. Tiles are handed out by an atomic ticket so a tile only ever waits on tiles
// that already started (forward progress without co-residency assumptions).
//   BLOCKS : false: item count = counts[visit[r]]; true: blocks touched by the rectangle in keys[r]
//            (keys = the depth-sorted keys, already in visiting order)
//   visit  : visiting order (Gaussian index at position r), or nullptr for identity
//   offsets: [n] exclusive prefix of counts[visit[r]]
//   total  : [1] 64-bit sum (M), written by the last tile
//   status : [num_tiles] zeroed; ticket: [1] zeroed
//   chunk_owner (BLOCKS, optional): chunk_owner[c] = visiting position whose items contain item c * chunk --
//            the emission kernel's CTA c starts there instead of searching the offsets (two ~22-step
//            dependent binary searches per CTA were most of bin_expand's 0.078 ms)
template <bool BLOCKS>
__device__ __forceinline__ void
scan_counts_body(uint32_t n, const uint32_t* __restrict__ counts, const uint64_t* __restrict__ keys,
                 const uint32_t* __restrict__ visit, uint32_t* __restrict__ offsets, uint64_t* __restrict__ total,
                 uint64_t* __restrict__ status, uint32_t* __restrict__ ticket, uint32_t* __restrict__ chunk_owner, uint32_t chunk,
                 uint32_t rank0, const uint64_t* __restrict__ init);

template <bool BLOCKS>
__global__ void __launch_bounds__(SCAN_THREADS)
scan_counts_kernel(uint32_t n, const uint32_t* __restrict__ counts, const uint64_t* __restrict__ keys,
                   const uint32_t* __restrict__ visit,
                   uint32_t* __restrict__ offsets, uint64_t* __restrict__ total,
                   uint64_t* __restrict__ status, uint32_t* __restrict__ ticket,
                   uint32_t* __restrict__ chunk_owner, uint32_t chunk,
                   uint32_t rank0, const uint64_t* __restrict__ init, const uint32_t* __restrict__ only_if) {
  // rank0, init (front-first depth order, second part): the scan covers the visiting positions [rank0, rank0 + n) and
  // starts from *init, the total the scan of the positions before them left; only_if: nothing to do when *only_if == 0
  pdl_launch_dependents();
  pdl_wait();
  if (only_if && *only_if == 0u) return;
  scan_counts_body<BLOCKS>(n, counts, keys, visit, offsets, total, status, ticket, chunk_owner, chunk, rank0, init);
}

// one tile (one ticket) of the scan: the body of scan_counts_kernel, also run by front_sort_kernel (front_sort.cuh)
template <bool BLOCKS>
__device__ __forceinline__ void
scan_counts_body(uint32_t n, const uint32_t* __restrict__ counts, const uint64_t* __restrict__ keys,
                 const uint32_t* __restrict__ visit, uint32_t* __restrict__ offsets, uint64_t* __restrict__ total,
                 uint64_t* __restrict__ status, uint32_t* __restrict__ ticket, uint32_t* __restrict__ chunk_owner, uint32_t chunk,
                 uint32_t rank0, const uint64_t* __restrict__ init) {
  keys += rank0;
  offsets += rank0;
  __shared__ uint32_t s_tile;
  __shared__ uint64_t s_warp[SCAN_THREADS / 32];
  __shared__ uint64_t s_prefix;
  if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
  __syncthreads();
  const uint32_t tile = s_tile;
  if ((uint64_t)tile * SCAN_TILE >= n) return;   // (front_sort_kernel has more CTAs than the scan has tiles)
  const uint32_t base = tile * SCAN_TILE + threadIdx.x * SCAN_ITEMS;

  uint32_t c[SCAN_ITEMS];
  uint32_t tsum = 0;
  const bool whole = base + SCAN_ITEMS <= n && (rank0 & 3u) == 0u;   // this thread's items are all inside (and aligned): 128-bit accesses
  if (BLOCKS && whole) {
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; k += 2) {
      const ulonglong2 kk = *reinterpret_cast<const ulonglong2*>(keys + base + k);
      c[k] = scan_block_count(kk.x);
      c[k + 1] = scan_block_count(kk.y);
    }
  } else {
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
      const uint32_t r = base + k;
      c[k] = 0;
      if (r < n) c[k] = BLOCKS ? scan_block_count(keys[r]) : counts[visit ? visit[r] : r];
    }
  }
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) tsum += c[k];  // < 2^32: one Gaussian covers at most 2^22 tiles, 8 of them 2^25
  // warp inclusive scan of the thread sums
  const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
  uint64_t incl = tsum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint64_t v = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= d) incl += v;
  }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  uint64_t warp_excl = 0, block_sum = 0;
#pragma unroll
  for (int w = 0; w < SCAN_THREADS / 32; ++w) {
    const uint64_t v = s_warp[w];
    if (w < warp) warp_excl += v;
    block_sum += v;
  }

  if (warp == 0) {
    // warp-wide look-back: lane l inspects predecessor tile - 1 - l; the walk ends at the nearest tile
    // that has published its inclusive prefix (tile -1 counts as a prefix of 0)
    uint64_t excl = 0;
    if (tile == 0) {
      excl = init ? *init : 0ull;
      if (lane == 0) st_relaxed_u64(status, LB_FLAG_PREFIX | (excl + block_sum));
    } else {
      if (lane == 0) st_relaxed_u64(status + tile, LB_FLAG_AGG | block_sum);
      int64_t p = (int64_t)tile - 1 - (int64_t)lane;
      while (true) {
        const uint64_t sv = p >= 0 ? ld_relaxed_u64(status + p) : LB_FLAG_PREFIX;
        const uint64_t flag = sv & LB_FLAG_MASK;
        const uint32_t ready = __ballot_sync(0xffffffffu, flag != 0);
        const uint32_t pref = __ballot_sync(0xffffffffu, flag == LB_FLAG_PREFIX);
        const uint32_t upto = pref ? (0xffffffffu >> (31 - (__ffs(pref) - 1))) : 0xffffffffu;   // lanes 0..first prefix
        if ((ready & upto) != upto) continue;   // a tile in the window holds an earlier ticket: it is running
        uint64_t v = ((upto >> lane) & 1u) ? (sv & LB_VALUE_MASK) : 0ull;
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
        excl += v;
        if (pref) break;
        p -= 32;
      }
      if (lane == 0) st_relaxed_u64(status + tile, LB_FLAG_PREFIX | (excl + block_sum));
    }
    if (lane == 0) {
      s_prefix = excl;
      if ((uint64_t)(tile + 1) * SCAN_TILE >= n) *total = excl + block_sum;
    }
  }
  __syncthreads();
  uint64_t run = s_prefix + warp_excl + (incl - tsum);
  if (whole) {
    uint32_t o = (uint32_t)run;   // valid when M < 2^32 (checked on the host)
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; k += 4) {
      const uint4 v = make_uint4(o, o + c[k], o + c[k] + c[k + 1], o + c[k] + c[k + 1] + c[k + 2]);
      *reinterpret_cast<uint4*>(offsets + base + k) = v;
      o = v.w + c[k + 3];
    }
  }
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    const uint32_t r = base + k;
    if (r < n) {
      if (!whole) offsets[r] = (uint32_t)run;
      if (BLOCKS && chunk_owner && c[k]) {
        const uint64_t first = (run + chunk - 1) / chunk;   // first chunk boundary at or after my first item
        if (first * chunk < run + c[k]) chunk_owner[first] = rank0 + r;   // c[k] <= 256 < chunk: at most one boundary
      }
    }
    run += c[k];
  }
}

}  // namespace pvg

// scan_dup.cuh -- stage a2: exclusive prefix scan of the per-Gaussian tile counts in
// visiting order, then emission of one (tile | depth) 64-bit key + Gaussian index per
// tile instance (PAPER.md:L61 tile-based rasterisation, L70 depth sort; S11).
#pragma once

#include "common.cuh"

namespace pvg {

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

// Single-pass chained scan with decoupled look-back. Warp-aggregated: per-thread
// serial sums -> warp shuffles -> one partial per warp -> block aggregate, which is
// published in a 64-bit status word (flag | value) and resolved against predecessor
// tiles. Tiles are handed out by an atomic ticket so a tile only ever waits on tiles
// that already started (forward progress without co-residency assumptions).
//   visit  : visiting order (Gaussian index at position r), or nullptr for identity
//   offsets: [n] exclusive prefix of counts[visit[r]]
//   total  : [1] 64-bit sum (M), written by the last tile
//   status : [num_tiles] zeroed; ticket: [1] zeroed
__global__ void __launch_bounds__(SCAN_THREADS)
scan_counts_kernel(uint32_t n, const uint32_t* __restrict__ counts, const uint32_t* __restrict__ visit,
                   uint32_t* __restrict__ offsets, uint64_t* __restrict__ total,
                   uint64_t* __restrict__ status, uint32_t* __restrict__ ticket) {
  __shared__ uint32_t s_tile;
  __shared__ uint64_t s_warp[SCAN_THREADS / 32];
  __shared__ uint64_t s_prefix;
  if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
  __syncthreads();
  const uint32_t tile = s_tile;
  const uint32_t base = tile * SCAN_TILE + threadIdx.x * SCAN_ITEMS;

  uint32_t c[SCAN_ITEMS];
  uint32_t tsum = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    const uint32_t r = base + k;
    c[k] = 0;
    if (r < n) c[k] = counts[visit ? visit[r] : r];
    tsum += c[k];  // < 2^32: one Gaussian covers at most 2^22 tiles, 8 of them 2^25
  }
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

  if (threadIdx.x == 0) {
    uint64_t excl = 0;
    if (tile == 0) {
      st_relaxed_u64(status, LB_FLAG_PREFIX | block_sum);
    } else {
      st_relaxed_u64(status + tile, LB_FLAG_AGG | block_sum);
      int64_t p = (int64_t)tile - 1;
      while (true) {
        const uint64_t s = ld_relaxed_u64(status + p);
        const uint64_t flag = s & LB_FLAG_MASK;
        if (flag == 0) continue;  // predecessor has a ticket, so it is running: spin
        excl += s & LB_VALUE_MASK;
        if (flag == LB_FLAG_PREFIX) break;
        --p;
      }
      st_relaxed_u64(status + tile, LB_FLAG_PREFIX | (excl + block_sum));
    }
    s_prefix = excl;
    if ((uint64_t)(tile + 1) * SCAN_TILE >= n) *total = excl + block_sum;
  }
  __syncthreads();
  uint64_t run = s_prefix + warp_excl + (incl - tsum);
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    const uint32_t r = base + k;
    if (r < n) offsets[r] = (uint32_t)run;  // valid when M < 2^32 (checked on the host)
    run += c[k];
  }
}

constexpr int DUP_THREADS = 256;
constexpr int DUP_ITEMS = 8;
constexpr int DUP_CHUNK = DUP_THREADS * DUP_ITEMS;
constexpr int DUP_SPAN = 2048;  // visiting positions cached in shared memory per chunk

// Instance-parallel emission: block b owns output instances [b*CHUNK, (b+1)*CHUNK), so
// the work per block is uniform no matter how skewed the per-Gaussian counts are (1 ..
// every tile) and every store is a fully coalesced 256 B (keys) / 128 B (values) line per
// warp. The owning visiting position of an instance is the last r with offsets[r] <= i,
// found by binary search (shared-memory copy of the chunk's offset span when it fits).
__global__ void __launch_bounds__(DUP_THREADS)
duplicate_kernel(uint32_t n, uint64_t M, const uint32_t* __restrict__ offsets,
                 const uint32_t* __restrict__ visit, const uint4* __restrict__ tileinfo,
                 uint32_t tiles_x, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  __shared__ uint32_t s_off[DUP_SPAN];
  __shared__ uint32_t s_lo, s_hi;
  const uint64_t i0 = (uint64_t)blockIdx.x * DUP_CHUNK;
  const uint64_t i1 = min(i0 + (uint64_t)DUP_CHUNK, M);  // exclusive
  if (threadIdx.x < 2) {
    // last r with offsets[r] <= target
    const uint32_t target = (uint32_t)(threadIdx.x == 0 ? i0 : i1 - 1);
    uint32_t lo = 0, hi = n;  // invariant: offsets[lo] <= target (offsets[0] = 0), answer in [lo, hi)
    while (hi - lo > 1) {
      const uint32_t mid = lo + ((hi - lo) >> 1);
      if (offsets[mid] <= target) lo = mid; else hi = mid;
    }
    if (threadIdx.x == 0) s_lo = lo; else s_hi = lo;
  }
  __syncthreads();
  const uint32_t r_lo = s_lo, r_hi = s_hi;
  const uint32_t span = r_hi - r_lo + 1;
  const bool cached = span <= DUP_SPAN;
  if (cached)
    for (uint32_t k = threadIdx.x; k < span; k += DUP_THREADS) s_off[k] = offsets[r_lo + k];
  __syncthreads();

#pragma unroll
  for (int k = 0; k < DUP_ITEMS; ++k) {
    const uint64_t i = i0 + (uint64_t)k * DUP_THREADS + threadIdx.x;
    if (i >= i1) break;
    const uint32_t target = (uint32_t)i;
    uint32_t lo = 0, hi = span;
    if (cached) {
      while (hi - lo > 1) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        if (s_off[mid] <= target) lo = mid; else hi = mid;
      }
    } else {
      while (hi - lo > 1) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        if (offsets[r_lo + mid] <= target) lo = mid; else hi = mid;
      }
    }
    const uint32_t r = r_lo + lo;
    const uint32_t off = cached ? s_off[lo] : offsets[r];
    const uint32_t g = visit ? visit[r] : r;
    const uint4 ti = tileinfo[g];
    const uint32_t j = target - off;          // < ti.w * rect height
    const uint32_t row = j / ti.y;
    const uint32_t col = j - row * ti.y;
    const uint32_t tile = ((ti.x >> 16) + row) * tiles_x + (ti.x & 0xFFFFu) + col;
    keys[i] = ((uint64_t)tile << 32) | ti.z;
    vals[i] = g;
  }
}

}  // namespace pvg

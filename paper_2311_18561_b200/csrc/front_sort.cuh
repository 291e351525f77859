// front_sort.cuh -- the front of a front-first frame (onesweep.cuh), ordered and scanned in ONE launch.
//
// With the first slab at 1/16 of the block entries the front is some ten thousand pairs: three radix passes and the
// scan over it are four launches of a few microseconds of work each, and each launch in a dependent chain costs about
// 6 us on the B200 whatever it does (launch, ticket, first loads, drain). The host knows the front's size F when it
// launches them (it has read preprocess's totals by then), so when the front's tiles fit the GPU at once it launches one
// grid of exactly that many CTAs which runs the passes and the scan back to back, with a grid-wide barrier between them:
// the same tiles, the same ranking, the same look-back, the same values as the separate launches.
// (One CTA sorting the whole front in its shared memory was tried first and lost: 71 us against 50 -- a single SM's
// issue rate is the bound there.)
#pragma once

#include "common.cuh"
#include "onesweep.cuh"
#include "scan_dup.cuh"

namespace pvg {

constexpr int FSORT_THREADS = 512;
constexpr int FSORT_ITEMS = 2;
constexpr int FSORT_TILE = FSORT_THREADS * FSORT_ITEMS;
static_assert(FSORT_THREADS == SCAN_THREADS, "the scan tiles are run by the same thread blocks");
static_assert(SCAN_TILE >= FSORT_TILE, "a grid of one CTA per sort tile covers the scan's tiles");

// The kernel is launched cooperatively (cudaLaunchAttributeCooperative; the host launches at most 2 CTAs per SM, which
// its launch bounds let fit): all CTAs of the grid are resident together, so a CTA that waits here waits for CTAs that are
// running. bar: zeroed; target = gridDim.x * (barriers so far).
__device__ __forceinline__ void grid_barrier(uint32_t* bar, uint32_t target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(bar, 1u);
    while (*reinterpret_cast<volatile uint32_t*>(bar) < target) __nanosleep(32);
    __threadfence();
  }
  __syncthreads();
}

// Arguments as depth_pass_kernel<.., false, true> (the front's class: region = its histogram region with the DepthCtl
// block, lookback = its look-back words, tickets = its four tickets) and scan_counts_kernel<true> (positions 0 .. F - 1).
// lb_rows: rows of the look-back layout per pass (class_lookback_rows in pvg_api.cu).
__global__ void __launch_bounds__(FSORT_THREADS, 2)
front_sort_kernel(uint64_t* __restrict__ keys_a, uint32_t* __restrict__ vals_a, uint64_t* __restrict__ keys_b,
                  uint32_t* __restrict__ vals_b, const uint32_t* __restrict__ region, uint64_t* __restrict__ lookback,
                  uint32_t lb_rows, uint32_t* __restrict__ tickets, uint32_t* __restrict__ bar,
                  uint32_t* __restrict__ offsets, uint64_t* __restrict__ total, uint64_t* __restrict__ status,
                  uint32_t* __restrict__ scan_ticket, uint32_t* __restrict__ chunk_owner, uint32_t chunk) {
  pdl_launch_dependents();
  pdl_wait();
  const DepthCtl* ctl = reinterpret_cast<const DepthCtl*>(region + DH_CTL);
  const uint32_t F = ctl->survivors;
  uint64_t* lb = lookback;
  uint32_t phase = 0;
#pragma unroll 1
  for (int p = 0; p < 3; ++p) {
    depth_pass_body<FSORT_THREADS, FSORT_ITEMS, DS_BITS, false, true>(keys_a, vals_a, keys_b, vals_b, F, p, ds_shift(p), ctl,
                                                                      region + p * DS_RADIX, lb, tickets + p);
    lb += (size_t)lb_rows << DS_BITS;
    grid_barrier(bar, gridDim.x * ++phase);
  }
  if (!ctl->skip[3]) {   // keys of 2^27 and beyond in the front: the top digit
    depth_pass_body<FSORT_THREADS, FSORT_ITEMS, DS_TOP_BITS, false, true>(keys_a, vals_a, keys_b, vals_b, F, 3, ds_shift(3), ctl,
                                                                          region + 3 * DS_RADIX, lb, tickets + 3);
    grid_barrier(bar, gridDim.x * ++phase);
  }
  const uint64_t* keys = ctl->final_side ? keys_b : keys_a;
  scan_counts_body<true>(F, nullptr, keys, nullptr, offsets, total, status, scan_ticket, chunk_owner, chunk, 0u, nullptr);
}

}  // namespace pvg

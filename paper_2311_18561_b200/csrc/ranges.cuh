// ranges.cuh -- stage a4: per-tile [begin, end) in the sorted instance list,
// range[tile] = [lower_bound(tile << 32), lower_bound((tile + 1) << 32)) (DESIGN.md a4).
#pragma once

#include "common.cuh"

namespace pvg {

// Thread i looks at the boundary between sorted keys i-1 and i. Tiles strictly between
// the two tile ids are empty and get begin == end == i, exactly as lower_bound would
// give; thread 0 also closes the tiles before the first key and thread M-1 those after
// the last. M == 0 is handled on the host (all ranges are [0,0)).
__global__ void __launch_bounds__(256)
tile_ranges_kernel(const uint64_t* __restrict__ keys, uint64_t M, uint32_t num_tiles,
                   uint2* __restrict__ ranges) {
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M) return;
  const uint32_t cur = (uint32_t)(__ldcs(keys + i) >> 32);
  if (i == 0) {
    for (uint32_t t = 0; t < cur; ++t) ranges[t] = make_uint2(0u, 0u);
    ranges[cur].x = 0u;
  } else {
    const uint32_t prev = (uint32_t)(keys[i - 1] >> 32);
    if (prev != cur) {
      ranges[prev].y = (uint32_t)i;
      for (uint32_t t = prev + 1; t < cur; ++t) ranges[t] = make_uint2((uint32_t)i, (uint32_t)i);
      ranges[cur].x = (uint32_t)i;
    }
  }
  if (i == M - 1) {
    ranges[cur].y = (uint32_t)M;
    for (uint32_t t = cur + 1; t < num_tiles; ++t) ranges[t] = make_uint2((uint32_t)M, (uint32_t)M);
  }
}

}  // namespace pvg

// tilebin.cuh -- per-tile instance counts without touching the instance list.
//
// Every surviving Gaussian adds +1 to each tile of its rectangle. Instead of M atomic
// increments (or a pass over the M sorted keys), tile_grid_kernel adds the rectangle's four
// corners to a 2-D difference array (4 integer atomics per Gaussian) and tile_prefix_kernel
// integrates it: a 2-D prefix sum gives the exact number of instances of every tile.
// From those counts follow, with no further HBM traffic,
//   * the per-tile ranges  range[tile] = [lower_bound(tile<<32), lower_bound((tile+1)<<32))
//     (stage a4: an exclusive scan of the counts in row-major tile order), and
//   * the digit histograms of the tile-id bits that the onesweep passes need (stage a3).
// Integer adds commute, so the result is deterministic and bit-exact.
#pragma once

#include "common.cuh"
#include "onesweep.cuh"

namespace pvg {

constexpr int TG_THREADS = 1024;

// The difference array. One persistent CTA per SM accumulates the four corner updates of its share
// of the rectangles in a shared-memory copy of the grid (they are heavily contended: clamped
// rectangles all hit the border cells) and then adds its non-zero cells to the global grid.
// use_smem = 0 (grid larger than shared memory): update the global grid directly.
__global__ void __launch_bounds__(TG_THREADS)
tile_grid_kernel(const uint4* __restrict__ tileinfo, uint32_t n, int TX, int TY, int use_smem, int* __restrict__ grid) {
  extern __shared__ int s_grid[];
  const int stride = tilegrid_stride(TX);
  const int cells = stride * (TY + 1);
  int* g = grid;
  if (use_smem) {
    for (int k = threadIdx.x; k < cells; k += TG_THREADS) s_grid[k] = 0;
    __syncthreads();
    g = s_grid;
  }
  for (uint32_t i = blockIdx.x * TG_THREADS + threadIdx.x; i < n; i += gridDim.x * TG_THREADS) {
    const uint4 ti = tileinfo[i];
    if (ti.w == 0u) continue;
    const int x0 = (int)(ti.x & 0xFFFFu), y0 = (int)(ti.x >> 16);
    tilegrid_add_rect(g, stride, x0, y0, x0 + (int)(ti.y & 0xFFFFu) - 1, y0 + (int)(ti.y >> 16) - 1);
  }
  if (use_smem) {
    __syncthreads();
    for (int k = threadIdx.x; k < cells; k += TG_THREADS) {
      const int v = s_grid[k];
      if (v) atomicAdd(grid + k, v);
    }
  }
}

constexpr int TB_THREADS = 1024;

// Single block. `grid` is the difference array in global memory ((TY+1) rows of `stride`
// ints); it is integrated in shared memory when it fits (use_smem) and in place otherwise.
// plan.shift[] are KEY bit positions (tile id sits at bit 32).
__global__ void __launch_bounds__(TB_THREADS)
tile_prefix_kernel(int* __restrict__ grid, int TX, int TY, int use_smem, const __grid_constant__ SortPlan plan,
                   uint2* __restrict__ ranges, uint32_t* __restrict__ hist /* [passes][256], exclusive */,
                   uint64_t* __restrict__ total_out) {
  extern __shared__ int s_dyn[];
  __shared__ uint32_t s_hist[OS_MAX_PASSES * OS_RADIX];
  __shared__ uint64_t s_part[TB_THREADS / 32];
  const int tid = threadIdx.x;
  const int stride = tilegrid_stride(TX);
  const int cells = stride * (TY + 1);
  int* g = grid;
  if (use_smem) {
    for (int k = tid; k < cells; k += TB_THREADS) s_dyn[k] = grid[k];
    g = s_dyn;
  }
  for (int k = tid; k < plan.num_passes * OS_RADIX; k += TB_THREADS) s_hist[k] = 0;
  __syncthreads();
  for (int row = tid; row <= TY; row += TB_THREADS) {   // prefix along x
    int run = 0;
    int* r = g + row * stride;
    for (int x = 0; x <= TX; ++x) { run += r[x]; r[x] = run; }
  }
  __syncthreads();
  for (int col = tid; col <= TX; col += TB_THREADS) {   // prefix along y
    int run = 0;
    for (int y = 0; y <= TY; ++y) { run += g[y * stride + col]; g[y * stride + col] = run; }
  }
  __syncthreads();
  // exclusive scan of the counts in row-major tile order: thread t owns a contiguous segment
  const uint32_t tiles = (uint32_t)TX * (uint32_t)TY;
  const uint32_t per = (tiles + TB_THREADS - 1) / TB_THREADS;
  const uint32_t t0 = min(tiles, (uint32_t)tid * per), t1 = min(tiles, t0 + per);
  uint64_t sum = 0;
  for (uint32_t tl = t0; tl < t1; ++tl) sum += (uint32_t)g[(tl / TX) * stride + (tl % TX)];
  const uint32_t lane = lane_id(), warp = tid >> 5;
  uint64_t incl = sum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint64_t v = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= d) incl += v;
  }
  if (lane == 31) s_part[warp] = incl;
  __syncthreads();
  uint64_t wex = 0, all = 0;
  for (int w = 0; w < TB_THREADS / 32; ++w) {
    const uint64_t v = s_part[w];
    if (w < (int)warp) wex += v;
    all += v;
  }
  uint64_t run = wex + incl - sum;
  for (uint32_t tl = t0; tl < t1; ++tl) {
    const uint32_t c = (uint32_t)g[(tl / TX) * stride + (tl % TX)];
    ranges[tl] = make_uint2((uint32_t)run, (uint32_t)(run + c));
    if (c)
      for (int p = 0; p < plan.num_passes; ++p) {
        const uint32_t d = (tl >> (plan.shift[p] - 32)) & ((1u << plan.bits[p]) - 1u);
        atomicAdd(&s_hist[p * OS_RADIX + d], c);
      }
    run += c;
  }
  if (tid == 0) *total_out = all;
  __syncthreads();
  // exclusive scan of each pass's histogram (256 threads per pass)
  for (int p = 0; p < plan.num_passes; ++p) {
    uint32_t v = 0, inc = 0;
    if (tid < OS_RADIX) {
      v = s_hist[p * OS_RADIX + tid];
      inc = v;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
      }
      if (lane == 31) s_part[warp] = inc;
    }
    __syncthreads();
    if (tid < OS_RADIX) {
      uint32_t wx = 0;
      for (uint32_t w = 0; w < warp; ++w) wx += (uint32_t)s_part[w];
      hist[p * OS_RADIX + tid] = wx + inc - v;
    }
    __syncthreads();
  }
}

}  // namespace pvg

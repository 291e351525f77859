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
// The same is done one level up for the 8x8-tile blocks of blockbin.cuh: a second, tiny
// difference array over the block grid gives the number of block entries per block, hence
// where each block's entries start after the split (bin_start) and how its list is cut into
// chunks (chunk_start) -- and the totals M and Mb that size the frame's buffers, early enough
// for the host to read them while the depth sort is still running.
// Integer adds commute, so the result is deterministic and bit-exact.
#pragma once

#include "common.cuh"
#include "onesweep.cuh"

namespace pvg {

constexpr int TG_THREADS = 1024;
constexpr int TB_MAX_BINS = 256;   // == BB_MAX_BINS (blockbin.cuh)
#ifndef PVG_BB_CHUNK
#define PVG_BB_CHUNK 512
#endif
constexpr int TB_CHUNK = PVG_BB_CHUNK;   // == BB_CHUNK

// Layout of the global grid buffer: the tile difference array, then the block difference array.
__host__ __device__ inline int tilegrid_cells(int tiles_x, int tiles_y) { return tilegrid_stride(tiles_x) * (tiles_y + 1); }
__host__ __device__ inline int blocks_of(int tiles) { return (tiles + 7) >> 3; }

// The difference arrays. One persistent CTA per SM accumulates the corner updates of its share
// of the rectangles in shared-memory copies of the grids (they are heavily contended: clamped
// rectangles all hit the border cells) and then adds its non-zero cells to the global grids.
// use_smem = 0 (grids larger than shared memory): update the global grids directly.
// with_blocks: also the block-level array (rectangle in units of 8x8-tile blocks).
__global__ void __launch_bounds__(TG_THREADS)
tile_grid_kernel(const uint4* __restrict__ tileinfo, uint32_t n, int TX, int TY, int use_smem, int with_blocks,
                 int* __restrict__ grid) {
  extern __shared__ int s_grid[];
  const int stride = tilegrid_stride(TX);
  const int cells = stride * (TY + 1);
  const int BX = blocks_of(TX), BY = blocks_of(TY);
  const int bstride = tilegrid_stride(BX);
  const int bcells = with_blocks ? bstride * (BY + 1) : 0;
  int* g = grid;
  if (use_smem) {
    for (int k = threadIdx.x; k < cells + bcells; k += TG_THREADS) s_grid[k] = 0;
    __syncthreads();
    g = s_grid;
  }
  int* gb = g + cells;
  uint32_t survivors = 0;
  for (uint32_t i = blockIdx.x * TG_THREADS + threadIdx.x; i < n; i += gridDim.x * TG_THREADS) {
    const uint4 ti = tileinfo[i];
    if (ti.w == 0u) continue;
    ++survivors;
    const int x0 = (int)(ti.x & 0xFFFFu), y0 = (int)(ti.x >> 16);
    const int x1 = x0 + (int)(ti.y & 0xFFFFu) - 1, y1 = y0 + (int)(ti.y >> 16) - 1;
    tilegrid_add_rect(g, stride, x0, y0, x1, y1);
    if (with_blocks) tilegrid_add_rect(gb, bstride, x0 >> 3, y0 >> 3, x1 >> 3, y1 >> 3);
  }
  if (use_smem) {
    __syncthreads();
    for (int k = threadIdx.x; k < cells + bcells; k += TG_THREADS) {
      const int v = s_grid[k];
      if (v) atomicAdd(grid + k, v);
    }
  }
  // number of surviving Gaussians S (a statistic for pvg_frame_stats): one extra cell after the grids
  survivors = __reduce_add_sync(0xffffffffu, survivors);
  if ((threadIdx.x & 31u) == 0 && survivors) atomicAdd(grid + cells + bcells, (int)survivors);
}

constexpr int TB_THREADS = 1024;

// in-place 2-D inclusive prefix sum of a (rows x cols) grid with row stride `stride`
__device__ __forceinline__ void grid_prefix_2d(int* g, int rows, int cols, int stride) {
  for (int row = threadIdx.x; row < rows; row += TB_THREADS) {
    int run = 0;
    int* r = g + row * stride;
    for (int x = 0; x < cols; ++x) { run += r[x]; r[x] = run; }
  }
  __syncthreads();
  for (int col = threadIdx.x; col < cols; col += TB_THREADS) {
    int run = 0;
    for (int y = 0; y < rows; ++y) { run += g[y * stride + col]; g[y * stride + col] = run; }
  }
  __syncthreads();
}

// Single block. `grid` holds the difference arrays in global memory; they are integrated in
// shared memory when they fit (use_smem) and in place otherwise.
// plan.shift[] are KEY bit positions (tile id sits at bit 32).
//   ranges[tile]            = [begin, end) of the tile in the sorted list
//   hist[pass][256]         = exclusive digit histograms of the tile-id passes
//   totals[0] = M (tile instances), totals[1] = Mb (block entries; with_blocks), totals[2] = S (survivors);
//   totals_host[0..2]: the same, in mapped host memory
//   bin_start[257], chunk_start[257] (with_blocks): see blockbin.cuh
// parts: bit 0 -- the tile level (ranges, hist, totals 0 and 2); bit 1 -- the block level (bin_start, chunk_start,
// totals 1). The two levels integrate different arrays: a front-first frame launches the block level first, on its own,
// because bin_emit waits for nothing else of this kernel (the ranges are first read by bin_write).
__global__ void __launch_bounds__(TB_THREADS)
tile_prefix_kernel(int* __restrict__ grid, int TX, int TY, int use_smem, int with_blocks, int parts, const __grid_constant__ SortPlan plan,
                   uint2* __restrict__ ranges, uint32_t* __restrict__ hist, uint64_t* __restrict__ totals,
                   uint32_t* __restrict__ bin_start, uint32_t* __restrict__ chunk_start,
                   volatile uint64_t* __restrict__ totals_host) {
  extern __shared__ int s_dyn[];
  __shared__ uint32_t s_hist[OS_MAX_PASSES * OS_RADIX];
  __shared__ uint64_t s_part[TB_THREADS / 32];
  __shared__ uint32_t s_a[TB_MAX_BINS / 32], s_b[TB_MAX_BINS / 32];
  const int tid = threadIdx.x;
  const int stride = tilegrid_stride(TX);
  const int cells = stride * (TY + 1);
  const int BX = blocks_of(TX), BY = blocks_of(TY);
  const int bstride = tilegrid_stride(BX);
  const int bcells = with_blocks ? bstride * (BY + 1) : 0;
  int* g = grid;
  if (use_smem) {
    const int k0 = (parts & 1) ? 0 : cells, k1 = (parts & 2) ? cells + bcells : cells;
    for (int k = k0 + tid; k < k1; k += TB_THREADS) s_dyn[k] = grid[k];
    g = s_dyn;
  }
  for (int k = tid; k < plan.num_passes * OS_RADIX; k += TB_THREADS) s_hist[k] = 0;
  __syncthreads();
  const uint32_t lane = lane_id(), warp = tid >> 5;
  if (parts & 1) {
  grid_prefix_2d(g, TY + 1, TX + 1, stride);
  // exclusive scan of the counts in row-major tile order: thread t owns a contiguous segment
  const uint32_t tiles = (uint32_t)TX * (uint32_t)TY;
  const uint32_t per = (tiles + TB_THREADS - 1) / TB_THREADS;
  const uint32_t t0 = min(tiles, (uint32_t)tid * per), t1 = min(tiles, t0 + per);
  uint64_t sum = 0;
  for (uint32_t tl = t0; tl < t1; ++tl) sum += (uint32_t)g[(tl / TX) * stride + (tl % TX)];
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
  // totals_host: the same three words in mapped pinned host memory, stored by this thread block itself -- a
  // copy-engine readback would queue behind the image copy of the previous frame (pvg_render_host_async)
  if (tid == 0) {
    const uint64_t surv = (uint32_t)grid[cells + bcells];
    totals[0] = all; totals[2] = surv;
    totals_host[0] = all; totals_host[2] = surv;
  }
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
  }   // parts & 1
  if (!with_blocks || !(parts & 2)) return;
  // block entries per block -> bin_start (exclusive scan) and chunk_start (scan of ceil(count / chunk))
  int* gb = g + cells;
  grid_prefix_2d(gb, BY + 1, BX + 1, bstride);
  if (tid < TB_MAX_BINS) {
    const uint32_t c = tid < BX * BY ? (uint32_t)gb[(tid / BX) * bstride + (tid % BX)] : 0u;
    const uint32_t k = (c + TB_CHUNK - 1) / TB_CHUNK;
    uint32_t ia = c, ib = k;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t ta = __shfl_up_sync(0xffffffffu, ia, d), tb = __shfl_up_sync(0xffffffffu, ib, d);
      if (lane >= d) { ia += ta; ib += tb; }
    }
    if (lane == 31) { s_a[warp] = ia; s_b[warp] = ib; }
    asm volatile("bar.sync 1, %0;" ::"n"(TB_MAX_BINS));
    uint32_t wa = 0, wb = 0;
    for (uint32_t w = 0; w < warp; ++w) { wa += s_a[w]; wb += s_b[w]; }
    bin_start[tid] = wa + ia - c;
    chunk_start[tid] = wb + ib - k;
    if (tid == TB_MAX_BINS - 1) {
      bin_start[TB_MAX_BINS] = wa + ia;
      chunk_start[TB_MAX_BINS] = wb + ib;
      totals[1] = wa + ia;
      totals_host[1] = wa + ia;
    }
  }
}

}  // namespace pvg

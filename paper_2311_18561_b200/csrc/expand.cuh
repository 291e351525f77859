// expand.cuh -- stage a2 (emission), lean version: one CTA owns EXP_CHUNK consecutive output
// instances. Instead of a binary search per instance (79 instructions per instance in the first
// version, profiles/r01), the owners of the chunk are staged once in shared memory, each owner
// marks the first instance it owns, and a max-scan spreads the owner index over the chunk;
// an instance then costs one small table lookup and a handful of integer operations.
// Output is either the 64-bit (tile | depth) key + Gaussian index, or the compact
// (u16 tile id, u32 Gaussian index) pair used when the depth bits are already in order.
#pragma once

#include "common.cuh"

namespace pvg {

constexpr int EXP_THREADS = 256;
constexpr int EXP_ITEMS = 16;
constexpr int EXP_CHUNK = EXP_THREADS * EXP_ITEMS;
constexpr int EXP_SPAN = 1024;  // owners staged per chunk; larger spans take the search path

struct ExpandSmem {
  int4 owner[EXP_SPAN];        // (first instance - chunk start, Gaussian, x0 | y0 << 16, rect width)
  float rcp[EXP_SPAN];         // 1 / rect width
  uint32_t zbits[EXP_SPAN];    // fp32 bits of the depth
  alignas(16) uint16_t own[EXP_CHUNK];  // owner slot of every instance of the chunk
  uint32_t warp_max[EXP_THREADS / 32];
  uint32_t lo, hi;
};

// last r in [0, n) with offsets[r] <= target (offsets[0] == 0)
__device__ __forceinline__ uint32_t last_owner_leq(const uint32_t* __restrict__ offsets, uint32_t n, uint32_t target) {
  uint32_t lo = 0, hi = n;
  while (hi - lo > 1) {
    const uint32_t mid = lo + ((hi - lo) >> 1);
    if (offsets[mid] <= target) lo = mid; else hi = mid;
  }
  return lo;
}

// tile id of the j-th tile (row-major inside the rectangle) of a rectangle at (x0,y0) of width w
__device__ __forceinline__ uint32_t rect_tile(uint32_t xy, uint32_t w, float rcp, uint32_t j, uint32_t tiles_x) {
  uint32_t row = __float2uint_rz(((float)j + 0.5f) * rcp);
  if (row * w > j) --row;                 // the float quotient is within one of the exact one
  else if ((row + 1) * w <= j) ++row;
  const uint32_t col = j - row * w;
  return ((xy >> 16) + row) * tiles_x + (xy & 0xFFFFu) + col;
}

// visit: visiting order (nullptr = identity). COMPACT: write tiles16/vals, else keys/vals.
template <bool COMPACT>
__global__ void __launch_bounds__(EXP_THREADS)
expand_kernel(uint32_t n, uint32_t M, const uint32_t* __restrict__ offsets, const uint32_t* __restrict__ visit,
              const uint4* __restrict__ tileinfo, uint32_t tiles_x, uint64_t* __restrict__ keys,
              uint16_t* __restrict__ tiles16, uint32_t* __restrict__ vals) {
  __shared__ ExpandSmem s;
  const uint32_t tid = threadIdx.x;
  const uint32_t i0 = blockIdx.x * EXP_CHUNK;
  const uint32_t i1 = min(i0 + (uint32_t)EXP_CHUNK, M);  // exclusive; M < 2^32 - EXP_CHUNK is checked on the host
  if (tid == 0) s.lo = last_owner_leq(offsets, n, i0);
  if (tid == 32) s.hi = last_owner_leq(offsets, n, i1 - 1);
  // clear the owner marks (16 u16 per thread)
  reinterpret_cast<uint4*>(s.own)[2 * tid] = make_uint4(0u, 0u, 0u, 0u);
  reinterpret_cast<uint4*>(s.own)[2 * tid + 1] = make_uint4(0u, 0u, 0u, 0u);
  __syncthreads();
  const uint32_t r_lo = s.lo, span = s.hi - r_lo + 1;

  if (span <= EXP_SPAN) {
    // stage the owners; each owner with a non-empty rectangle marks its first instance
    for (uint32_t k = tid; k < span; k += EXP_THREADS) {
      const uint32_t r = r_lo + k;
      const uint32_t g = visit ? visit[r] : r;
      const uint4 ti = tileinfo[g];
      const int start = (int)(offsets[r] - i0);   // negative only for the owner that began before the chunk
      s.owner[k] = make_int4(start, (int)g, (int)ti.x, (int)(ti.y & 0xFFFFu));
      s.rcp[k] = 1.0f / (float)(ti.y & 0xFFFFu);
      s.zbits[k] = ti.z;
      if (ti.w != 0u && start < EXP_CHUNK) s.own[max(start, 0)] = (uint16_t)k;
    }
    __syncthreads();
    // max-scan of the marks: every instance gets the slot of the last owner that started at or before it
    uint4 a = reinterpret_cast<uint4*>(s.own)[2 * tid], b = reinterpret_cast<uint4*>(s.own)[2 * tid + 1];
    uint32_t w16[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
    uint32_t run = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) run = max(run, max(w16[q] & 0xFFFFu, w16[q] >> 16));
    uint32_t incl = run;
    const uint32_t lane = tid & 31u, warp = tid >> 5;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
      if (lane >= d) incl = max(incl, v);
    }
    if (lane == 31) s.warp_max[warp] = incl;
    uint32_t carry = __shfl_up_sync(0xffffffffu, incl, 1);
    if (lane == 0) carry = 0;
    __syncthreads();
    for (uint32_t wv = 0; wv < warp; ++wv) carry = max(carry, s.warp_max[wv]);
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const uint32_t lo16 = max(carry, w16[q] & 0xFFFFu);
      const uint32_t hi16 = max(lo16, w16[q] >> 16);
      carry = hi16;
      w16[q] = lo16 | (hi16 << 16);
    }
    reinterpret_cast<uint4*>(s.own)[2 * tid] = make_uint4(w16[0], w16[1], w16[2], w16[3]);
    reinterpret_cast<uint4*>(s.own)[2 * tid + 1] = make_uint4(w16[4], w16[5], w16[6], w16[7]);
    __syncthreads();
    // emit: thread-strided so that every warp store is one contiguous line
#pragma unroll 4
    for (int k = 0; k < EXP_ITEMS; ++k) {
      const uint32_t p = k * EXP_THREADS + tid;
      if (i0 + p >= i1) break;
      const uint32_t slot = s.own[p];
      const int4 o = s.owner[slot];
      const uint32_t tile = rect_tile((uint32_t)o.z, (uint32_t)o.w, s.rcp[slot], (uint32_t)((int)p - o.x), tiles_x);
      if (COMPACT) tiles16[i0 + p] = (uint16_t)tile;
      else keys[i0 + p] = ((uint64_t)tile << 32) | s.zbits[slot];
      vals[i0 + p] = (uint32_t)o.y;
    }
  } else {
    // many tiny rectangles in one chunk: binary search per instance over the global offsets
    for (int k = 0; k < EXP_ITEMS; ++k) {
      const uint32_t p = k * EXP_THREADS + tid;
      if (i0 + p >= i1) break;
      uint32_t lo = 0, hi = span;
      while (hi - lo > 1) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        if (offsets[r_lo + mid] <= i0 + p) lo = mid; else hi = mid;
      }
      const uint32_t r = r_lo + lo;
      const uint32_t g = visit ? visit[r] : r;
      const uint4 ti = tileinfo[g];
      const uint32_t rw = ti.y & 0xFFFFu;
      const uint32_t tile = rect_tile(ti.x, rw, 1.0f / (float)rw, i0 + p - offsets[r], tiles_x);
      if (COMPACT) tiles16[i0 + p] = (uint16_t)tile;
      else keys[i0 + p] = ((uint64_t)tile << 32) | ti.z;
      vals[i0 + p] = g;
    }
  }
}

}  // namespace pvg

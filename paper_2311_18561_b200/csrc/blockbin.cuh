// blockbin.cuh -- stages a2 + a3 (instance part) for depth-presorted Gaussians, without ever
// materialising or ranking the M individual (tile | depth) keys.
//
// The sorted instance list of DESIGN.md S11 is, tile by tile, "the Gaussians whose rectangle
// covers the tile, in depth order" (PAPER.md:L61 tiles, L70 depth sort). Once the Gaussians are
// in depth order (the n-key onesweep sort), that list can be produced with one ranked item per
// (Gaussian, 8x8-tile block) instead of one per (Gaussian, tile) -- 30x fewer at 1920x1280:
//   1. bin_expand: every Gaussian emits, in depth order, one ENTRY per block its rectangle
//      touches: (block id, Gaussian index, 64-bit mask of the block's tiles it covers);
//   2. bin_pass: ONE stable onesweep digit pass splits the entries by block id (<= 256 blocks);
//      inside a block the entries stay in depth order;
//      (1 and 2 run as ONE kernel, bin_emit_kernel: the CTA that ranks a tile of entries forms them
//      in registers, so the unsplit entries never exist in HBM; the two-kernel form is kept behind
//      PVG_BIN_FUSED=0)
//   (the entries per block, hence bin_start / chunk_start, come from tilebin.cuh's block grid)
//   3. bin_write: a warp owns (chunk of 512 entries of a block, 32 of the block's tiles). It counts
//      how many of its entries cover each tile, and a decoupled look-back over the block's earlier
//      chunks, started at the tile's range begin (tilebin.cuh), gives its write position in every
//      tile list. Then, with a lane holding one entry, one ballot of "covers it" per tile ranks 32
//      entries, and the covering lanes store their Gaussian index as one contiguous run of that
//      tile's list.
// The result is bit-identical to the stable LSD sort of the 64-bit keys: within a tile the
// order is (depth bits, index), exactly the visiting order of the entries.
#pragma once

#include "common.cuh"
#include "onesweep.cuh"

namespace pvg {

constexpr int BB_MAX_BINS = 256;  // one 8-bit digit pass
#ifndef PVG_BB_CHUNK
#define PVG_BB_CHUNK 512
#endif
constexpr int BB_CHUNK = PVG_BB_CHUNK;   // entries per (warp pair) chunk of the write walk (tilebin.cuh cuts the lists)

__host__ __device__ inline uint32_t bb_blocks(uint32_t tiles) { return (tiles + 7u) >> 3; }

// ---- 1. entry emission ---------------------------------------------------------------------
constexpr int BE_THREADS = 256;
constexpr int BE_ITEMS = 8;
constexpr int BE_CHUNK = BE_THREADS * BE_ITEMS;
constexpr int BE_SPAN = BE_CHUNK + 64;  // survivors come first in depth order and own >= 1 entry each

struct BinExpandSmem {
  int4 owner[BE_SPAN];                  // (first entry - chunk start, Gaussian, x0 | y0 << 16, x1 | y1 << 16)
  alignas(16) uint16_t own[BE_CHUNK];   // owner slot of every entry of the chunk
  uint32_t warp_max[BE_THREADS / 32];
  uint32_t lo, hi;
};

// entry j (row-major over the blocks of the rectangle) of a Gaussian: block id and tile mask
__device__ __forceinline__ void bb_entry(uint32_t xy0, uint32_t xy1, uint32_t j, uint32_t blocks_x,
                                         uint32_t& bin, uint64_t& mask) {
  const uint32_t x0 = xy0 & 0xFFFFu, y0 = xy0 >> 16, x1 = xy1 & 0xFFFFu, y1 = xy1 >> 16;
  const uint32_t bx0 = x0 >> 3, bw = (x1 >> 3) - bx0 + 1u;
  // j < 2^16, bw <= 2^8: (j + 0.5) / bw is at least 1/(2 bw) away from an integer, far more than
  // the rounding of the product, so the truncation is the exact quotient
  const uint32_t brow = __float2uint_rz(((float)j + 0.5f) * __frcp_rn((float)bw));
  const uint32_t bx = bx0 + (j - brow * bw), by = (y0 >> 3) + brow;
  bin = by * blocks_x + bx;
  const uint32_t lx0 = max(x0, bx * 8u) - bx * 8u, lx1 = min(x1, bx * 8u + 7u) - bx * 8u;
  const uint32_t ly0 = max(y0, by * 8u) - by * 8u, ly1 = min(y1, by * 8u + 7u) - by * 8u;
  const uint32_t rowmask = ((2u << (lx1 - lx0)) - 1u) << lx0;   // bits lx0..lx1 of one tile row
  const uint32_t nrows = ly1 - ly0 + 1u;
  const uint64_t rows = nrows == 8u ? ~0ull : (((1ull << (8u * nrows)) - 1ull) << (8u * ly0));
  mask = ((uint64_t)rowmask * 0x0101010101010101ull) & rows;    // bit (ty & 7) * 8 + (tx & 7)
}

// P13: clears from an entry's mask the tiles of the block that the
// Gaussian's region { alpha >= 1/255 } cannot reach. Per tile row the region's x-extent inside the band of pixel-centre
// rows is an interval (the ellipse's right / left boundary at the dy of the band nearest to where it peaks); tiles whose
// box of pixel centres misses it go. Integer work: every float operation is an individually rounded fp32 one
// (__f*_rn: no contraction), in the order the oracle's exact_row_span takes them, so both sides decide identically.
// r0 = (mx, my, z, o~), r1 = (a, b, c, hx) of the fp32 record.
static __device__ __noinline__ uint64_t bb_refine_mask(uint64_t mask, uint32_t bx, uint32_t by, float4 r0, float4 r1) {
  const float a = r1.x, b = r1.y, c = r1.z, hx = r1.w;
  const float det = __fsub_rn(__fmul_rn(a, c), __fmul_rn(b, b));
  const float k = __fdiv_rn(__fmul_rn(__fmul_rn(hx, hx), det), c);
  const float kk = __fadd_rn(__fmul_rn(k, 1.0002f), 2e-5f);
  const float dxm = __fsqrt_rn(__fdiv_rn(__fmul_rn(kk, c), det));
  const float dyr = -__fmul_rn(__fdiv_rn(b, c), dxm);
  const float ia = __fdiv_rn(1.0f, a);
  const float akk = __fmul_rn(a, kk);
  const float big = 3.0e38f;
  const bool refine = (det > 0.0f) && (a > 0.0f) && (c > 0.0f) && (fabsf(kk) <= big) && (fabsf(dxm) <= big) && (fabsf(ia) <= big) &&
                      (fabsf(dyr) <= big) && (kk > 0.0f);
  if (!refine) return mask;
#pragma unroll 1
  for (uint32_t ly = 0; ly < 8u; ++ly) {
    const uint32_t row = (uint32_t)(mask >> (8u * ly)) & 0xFFu;
    if (!row) continue;
    const int ty = (int)(by * 8u + ly);
    const float y0 = __fsub_rn(__fadd_rn((float)(16 * ty), 0.5f), r0.y), y1 = __fadd_rn(y0, 15.0f);
    uint32_t keep = row;
    if ((y0 > 0.0f && __fsub_rn(akk, __fmul_rn(__fmul_rn(det, y0), y0)) < 0.0f) ||
        (y1 < 0.0f && __fsub_rn(akk, __fmul_rn(__fmul_rn(det, y1), y1)) < 0.0f)) {
      keep = 0u;
    } else {
      const float tr = fminf(fmaxf(dyr, y0), y1), tl = fminf(fmaxf(-dyr, y0), y1);
      const float dr = fmaxf(__fsub_rn(akk, __fmul_rn(__fmul_rn(det, tr), tr)), 0.0f);
      const float dl = fmaxf(__fsub_rn(akk, __fmul_rn(__fmul_rn(det, tl), tl)), 0.0f);
      const float xr = __fmul_rn(__fsub_rn(__fsqrt_rn(dr), __fmul_rn(b, tr)), ia);
      const float xl = __fmul_rn(__fsub_rn(-__fsqrt_rn(dl), __fmul_rn(b, tl)), ia);
      const float XR = __fadd_rn(__fadd_rn(r0.x, xr), 1e-3f), XL = __fsub_rn(__fadd_rn(r0.x, xl), 1e-3f);
      if (fabsf(XR) <= big && fabsf(XL) <= big) {
        const float fh = floorf(__fmul_rn(__fsub_rn(XR, 0.5f), 0.0625f)), fl = ceilf(__fmul_rn(__fsub_rn(XL, 15.5f), 0.0625f));
        const int h = (int)fminf(fmaxf(fh, -2.0f), 1.0e6f), l = (int)fminf(fmaxf(fl, -2.0f), 1.0e6f);
        // columns [l, h] of the image -> bits of this block's row
        const int lo = max(l - (int)(bx * 8u), 0), hi = min(h - (int)(bx * 8u), 7);
        keep = lo <= hi ? (row & (((2u << hi) - 1u) & ~((1u << lo) - 1u))) : 0u;
      }
    }
    mask &= ~((uint64_t)(row & ~keep) << (8u * ly));
  }
  return mask;
}

// One CTA owns BE_CHUNK consecutive entries. The owners of the chunk are staged in shared
// memory, each marks its first entry, and a max-scan spreads the owner slot over the chunk
// (same scheme as expand.cuh). keys/visit: the depth-sorted (rect | depth, Gaussian) pairs;
// boffsets: exclusive scan of the blocks touched, in that order.
__global__ void __launch_bounds__(BE_THREADS)
bin_expand_kernel(uint32_t n, uint32_t Mb, const uint32_t* __restrict__ boffsets, const uint32_t* __restrict__ chunk_owner,
                  const uint64_t* __restrict__ keys, const uint32_t* __restrict__ visit, uint32_t blocks_x, uint8_t* __restrict__ e_bin,
                  uint32_t* __restrict__ e_g, uint64_t* __restrict__ e_mask) {
  __shared__ BinExpandSmem s;
  const uint32_t tid = threadIdx.x;
  const uint32_t i0 = blockIdx.x * BE_CHUNK;
  const uint32_t i1 = min(i0 + (uint32_t)BE_CHUNK, Mb);
  if (tid == 0) {
    // owners of the chunk: from the one that contains its first entry (written by the scan) to the one that
    // contains the next chunk's first entry; the last chunk stages up to the span limit (owners that start
    // beyond the chunk leave no mark)
    const uint32_t lo = chunk_owner[blockIdx.x];
    s.lo = lo;
    s.hi = (uint64_t)(blockIdx.x + 1) * BE_CHUNK < Mb ? chunk_owner[blockIdx.x + 1] : min(lo + (uint32_t)BE_SPAN, n) - 1u;
  }
  reinterpret_cast<uint4*>(s.own)[tid] = make_uint4(0u, 0u, 0u, 0u);   // 8 u16 per thread
  __syncthreads();
  const uint32_t r_lo = s.lo, span = s.hi - r_lo + 1u;

  if (span <= BE_SPAN) {
    for (uint32_t k = tid; k < span; k += BE_THREADS) {
      const uint32_t r = r_lo + k;
      const uint64_t key = keys[r];
      const uint32_t rc = (uint32_t)(key >> 32);   // (x0, y0, x1, y1), 8 bits each
      const int start = (int)(boffsets[r] - i0);   // negative only for the owner that began before the chunk
      s.owner[k] = make_int4(start, (int)visit[r], (int)((rc & 0xFFu) | ((rc & 0xFF00u) << 8)),
                             (int)(((rc >> 16) & 0xFFu) | ((rc >> 24) << 16)));
      if ((uint32_t)key != 0xFFFFFFFFu && start < BE_CHUNK) s.own[max(start, 0)] = (uint16_t)k;
    }
    __syncthreads();
    // inclusive max-scan of the marks (slot numbers increase along the chunk)
    const uint4 a = reinterpret_cast<uint4*>(s.own)[tid];
    uint32_t w16[4] = {a.x, a.y, a.z, a.w};
    uint32_t run = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) run = max(run, max(w16[q] & 0xFFFFu, w16[q] >> 16));
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
    for (int q = 0; q < 4; ++q) {
      const uint32_t lo16 = max(carry, w16[q] & 0xFFFFu);
      const uint32_t hi16 = max(lo16, w16[q] >> 16);
      carry = hi16;
      w16[q] = lo16 | (hi16 << 16);
    }
    reinterpret_cast<uint4*>(s.own)[tid] = make_uint4(w16[0], w16[1], w16[2], w16[3]);
    __syncthreads();
#pragma unroll 4
    for (int k = 0; k < BE_ITEMS; ++k) {
      const uint32_t p = k * BE_THREADS + tid;
      if (i0 + p >= i1) break;
      const int4 o = s.owner[s.own[p]];
      uint32_t bin;
      uint64_t mask;
      bb_entry((uint32_t)o.z, (uint32_t)o.w, (uint32_t)((int)p - o.x), blocks_x, bin, mask);
      e_bin[i0 + p] = (uint8_t)bin;
      e_g[i0 + p] = (uint32_t)o.y;
      e_mask[i0 + p] = mask;
    }
  } else {
    // owners without entries inside the chunk (never the case in depth order): search per entry
    for (int k = 0; k < BE_ITEMS; ++k) {
      const uint32_t p = k * BE_THREADS + tid;
      if (i0 + p >= i1) break;
      uint32_t lo = 0, hi = span;
      while (hi - lo > 1) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        if (boffsets[r_lo + mid] <= i0 + p) lo = mid; else hi = mid;
      }
      const uint32_t r = r_lo + lo;
      const uint32_t g = visit[r];
      const uint32_t rc = (uint32_t)(keys[r] >> 32);
      uint32_t bin;
      uint64_t mask;
      bb_entry((rc & 0xFFu) | ((rc & 0xFF00u) << 8), ((rc >> 16) & 0xFFu) | ((rc >> 24) << 16), i0 + p - boffsets[r], blocks_x,
               bin, mask);
      e_bin[i0 + p] = (uint8_t)bin;
      e_g[i0 + p] = g;
      e_mask[i0 + p] = mask;
    }
  }
}

// ---- 2. stable split of the entries by block id ---------------------------------------------
#ifndef PVG_BP_THREADS
#define PVG_BP_THREADS 512   // cfg 3, fused: 512 x 8 0.128 ms, 256 x 16 0.132, 384 x 8 0.134, 256 x 8 (3 CTAs/SM) 0.143
#define PVG_BP_ITEMS 8
#define PVG_BP_MINB 2
#endif
constexpr int BP_THREADS = PVG_BP_THREADS;
constexpr int BP_ITEMS = PVG_BP_ITEMS;   // a multiple of 8

template <int BITS>
struct BinPassSmem {
  typename RadixCore<BP_THREADS, BP_ITEMS, BITS>::Smem core;
  uint64_t mask[BP_THREADS * BP_ITEMS];
  uint32_t g[BP_THREADS * BP_ITEMS];
  uint8_t bin[BP_THREADS * BP_ITEMS];
};

// One onesweep digit pass (RadixCore, decoupled look-back) over (block id; Gaussian, mask).
// The block id itself is not written: bin_start[] says where each block's entries live.
template <int BITS>
__global__ void __launch_bounds__(BP_THREADS, PVG_BP_MINB)
bin_pass_kernel(const uint8_t* __restrict__ bin_in, const uint32_t* __restrict__ g_in, const uint64_t* __restrict__ mask_in,
                uint32_t* __restrict__ g_out, uint64_t* __restrict__ mask_out, uint32_t n,
                const uint32_t* __restrict__ bin_start, uint64_t* __restrict__ lookback, uint32_t* __restrict__ ticket) {
  using Core = RadixCore<BP_THREADS, BP_ITEMS, BITS>;
  constexpr int TILE = Core::TILE;
  constexpr uint32_t MASK = (1u << BITS) - 1u;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  BinPassSmem<BITS>& s = *reinterpret_cast<BinPassSmem<BITS>*>(smem_raw);

  const uint32_t tile = Core::take_ticket(s.core, ticket);
  const uint32_t tile_base = tile * TILE;
  const uint32_t tile_n = min((uint32_t)TILE, n - tile_base);
  const uint32_t tid = threadIdx.x;
  const uint32_t wbase = (tid >> 5) * (BP_ITEMS * 32) + (tid & 31u);
  uint32_t dp[BP_ITEMS], g[BP_ITEMS];
  uint64_t mk[BP_ITEMS];
#pragma unroll
  for (int j = 0; j < BP_ITEMS; ++j) {
    const bool ok = wbase + j * 32 < tile_n;
    const uint32_t i = tile_base + wbase + j * 32;
    dp[j] = ok ? (uint32_t)__ldcs(bin_in + i) & MASK : MASK;   // block ids < 2^BITS; padding ranks last
    g[j] = ok ? __ldcs(g_in + i) : 0u;
    mk[j] = ok ? __ldcs(mask_in + i) : 0ull;
  }
  Core::rank(s.core, tile, dp, bin_start, lookback);
#pragma unroll
  for (int j = 0; j < BP_ITEMS; ++j) {
    s.bin[dp[j] >> 8] = (uint8_t)dp[j];   // rank() keeps the digit in the low 8 bits
    s.g[dp[j] >> 8] = g[j];
    s.mask[dp[j] >> 8] = mk[j];
  }
  __syncthreads();
  for (uint32_t p = tid; p < tile_n; p += BP_THREADS) {
    const uint32_t o = s.core.out_base[s.bin[p] & MASK] + p;
    g_out[o] = s.g[p];
    mask_out[o] = s.mask[p];
  }
}

// ---- 1 + 2 fused: the entries of a tile are formed in registers and split at once ------------
// bin_expand writes 13 B per entry only for bin_pass to read them back. Here the CTA that ranks a tile of
// BP_THREADS * BP_ITEMS entries forms them itself: the owners are staged as in bin_expand_kernel, every
// thread derives its BP_ITEMS entries (warp-striped, the order RadixCore ranks in), and the staging arrays of
// the split then reuse the shared memory of the owner table.
constexpr int BF_TILE = BP_THREADS * BP_ITEMS;
static_assert(BF_TILE == PVG_EMIT_TILE, "lazy_emit_first (common.cuh) counts bin_emit tiles");
constexpr int BF_SPAN = BF_TILE + 64;

template <int BITS>
struct BinEmitSmem {
  typename RadixCore<BP_THREADS, BP_ITEMS, BITS>::Smem core;
  uint32_t warp_max[BP_THREADS / 32];
  uint32_t lo, hi;
  union {
    struct {
      int4 owner[BF_SPAN];
      alignas(16) uint16_t own[BF_TILE];
    } a;
    struct {
      uint64_t mask[BF_TILE];
      uint32_t g[BF_TILE];
      uint8_t bin[BF_TILE];
    } b;
  };
};

// One tile of BF_TILE entries (the next ticket). Returns false, doing nothing, when the ticket is at or beyond
// tile_end (tile_end != 0 only in a launch whose CTAs loop over tickets).
template <int BITS, bool EXACT>
__device__ __forceinline__ bool
bin_emit_tile(BinEmitSmem<BITS>& s, uint32_t n, uint32_t Mb, const uint32_t* __restrict__ boffsets, const uint32_t* __restrict__ chunk_owner,
              const uint64_t* __restrict__ keys, const uint32_t* __restrict__ visit, uint32_t blocks_x,
              uint32_t* __restrict__ g_out, uint64_t* __restrict__ mask_out, const uint32_t* __restrict__ bin_start,
              uint64_t* __restrict__ lookback, uint32_t* __restrict__ ticket, const float4* __restrict__ record, uint32_t tile_end) {
  using Core = RadixCore<BP_THREADS, BP_ITEMS, BITS>;
  constexpr uint32_t MASK = (1u << BITS) - 1u;
  const uint32_t tile = Core::take_ticket(s.core, ticket);
  if (tile_end && tile >= tile_end) return false;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t i0 = tile * BF_TILE;
  const uint32_t tile_n = min((uint32_t)BF_TILE, Mb - i0);
  if (tid == 0) {
    const uint32_t lo = chunk_owner[tile];
    s.lo = lo;
    s.hi = (uint64_t)(tile + 1) * BF_TILE < Mb ? chunk_owner[tile + 1] : min(lo + (uint32_t)BF_SPAN, n) - 1u;
  }
  constexpr int OV = BP_ITEMS / 8;   // uint4 (8 u16 marks) per thread
#pragma unroll
  for (int q = 0; q < OV; ++q) reinterpret_cast<uint4*>(s.a.own)[OV * tid + q] = make_uint4(0u, 0u, 0u, 0u);
  __syncthreads();
  const uint32_t r_lo = s.lo, span = s.hi - r_lo + 1u;
  const uint32_t wbase = warp * (BP_ITEMS * 32) + lane;
  uint32_t dp[BP_ITEMS], g[BP_ITEMS];
  uint64_t mk[BP_ITEMS];

  if (span <= BF_SPAN) {
    for (uint32_t k = tid; k < span; k += BP_THREADS) {
      const uint32_t r = r_lo + k;
      const uint64_t key = keys[r];
      const uint32_t rc = (uint32_t)(key >> 32);   // (x0, y0, x1, y1), 8 bits each
      const int start = (int)(boffsets[r] - i0);   // negative only for the owner that began before the tile
      s.a.owner[k] = make_int4(start, (int)visit[r], (int)((rc & 0xFFu) | ((rc & 0xFF00u) << 8)),
                               (int)(((rc >> 16) & 0xFFu) | ((rc >> 24) << 16)));
      if ((uint32_t)key != 0xFFFFFFFFu && start < BF_TILE) s.a.own[max(start, 0)] = (uint16_t)k;
    }
    __syncthreads();
    // inclusive max-scan of the marks (slot numbers increase along the tile)
    uint32_t w16[4 * OV];
#pragma unroll
    for (int q = 0; q < OV; ++q) {
      const uint4 a = reinterpret_cast<uint4*>(s.a.own)[OV * tid + q];
      w16[4 * q] = a.x; w16[4 * q + 1] = a.y; w16[4 * q + 2] = a.z; w16[4 * q + 3] = a.w;
    }
    uint32_t run = 0;
#pragma unroll
    for (int q = 0; q < 4 * OV; ++q) run = max(run, max(w16[q] & 0xFFFFu, w16[q] >> 16));
    uint32_t incl = run;
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
    for (int q = 0; q < 4 * OV; ++q) {
      const uint32_t lo16 = max(carry, w16[q] & 0xFFFFu);
      const uint32_t hi16 = max(lo16, w16[q] >> 16);
      carry = hi16;
      w16[q] = lo16 | (hi16 << 16);
    }
#pragma unroll
    for (int q = 0; q < OV; ++q)
      reinterpret_cast<uint4*>(s.a.own)[OV * tid + q] = make_uint4(w16[4 * q], w16[4 * q + 1], w16[4 * q + 2], w16[4 * q + 3]);
    __syncthreads();
#pragma unroll
    for (int j = 0; j < BP_ITEMS; ++j) {
      const uint32_t p = wbase + j * 32;
      dp[j] = MASK; g[j] = 0u; mk[j] = 0ull;   // padding ranks last
      if (p < tile_n) {
        const int4 o = s.a.owner[s.a.own[p]];
        bb_entry((uint32_t)o.z, (uint32_t)o.w, (uint32_t)((int)p - o.x), blocks_x, dp[j], mk[j]);
        g[j] = (uint32_t)o.y;
      }
    }
  } else {
    // owners without entries inside the tile (never the case in depth order): search per entry
#pragma unroll
    for (int j = 0; j < BP_ITEMS; ++j) {
      const uint32_t p = wbase + j * 32;
      dp[j] = MASK; g[j] = 0u; mk[j] = 0ull;
      if (p < tile_n) {
        uint32_t lo = 0, hi = span;
        while (hi - lo > 1) {
          const uint32_t mid = lo + ((hi - lo) >> 1);
          if (boffsets[r_lo + mid] <= i0 + p) lo = mid; else hi = mid;
        }
        const uint32_t r = r_lo + lo;
        const uint32_t rc = (uint32_t)(keys[r] >> 32);
        bb_entry((rc & 0xFFu) | ((rc & 0xFF00u) << 8), ((rc >> 16) & 0xFFu) | ((rc >> 24) << 16), i0 + p - boffsets[r],
                 blocks_x, dp[j], mk[j]);
        g[j] = visit[r];
      }
    }
  }
  if (EXACT) {
#pragma unroll
    for (int j = 0; j < BP_ITEMS; ++j)
      if (mk[j]) {
        const float4 r0 = __ldg(record + 3 * (size_t)g[j]), r1 = __ldg(record + 3 * (size_t)g[j] + 1);
        mk[j] = bb_refine_mask(mk[j], dp[j] % blocks_x, dp[j] / blocks_x, r0, r1);
      }
  }
  __syncthreads();   // the owner table is dead: s.b reuses it
  Core::rank(s.core, tile, dp, bin_start, lookback);
#pragma unroll
  for (int j = 0; j < BP_ITEMS; ++j) {
    s.b.bin[dp[j] >> 8] = (uint8_t)dp[j];   // rank() keeps the digit in the low 8 bits
    s.b.g[dp[j] >> 8] = g[j];
    s.b.mask[dp[j] >> 8] = mk[j];
  }
  __syncthreads();
  for (uint32_t p = tid; p < tile_n; p += BP_THREADS) {
    const uint32_t o = s.core.out_base[s.b.bin[p] & MASK] + p;
    g_out[o] = s.b.g[p];
    mask_out[o] = s.b.mask[p];
  }
  return true;
}

// tile_end == 0: one tile per CTA (the grid is the number of tiles of the launch). tile_end != 0: the CTAs loop over
// tickets until they reach tile_end -- the second-round launch of the lazy lists, which usually finds nothing to do
// (*only_if == 0) and should then cost a few hundred CTAs, not thousands.
template <int BITS, bool EXACT>
__global__ void __launch_bounds__(BP_THREADS, PVG_BP_MINB)
bin_emit_kernel(uint32_t n, uint32_t Mb, const uint32_t* __restrict__ boffsets, const uint32_t* __restrict__ chunk_owner,
                const uint64_t* __restrict__ keys, const uint32_t* __restrict__ visit, uint32_t blocks_x,
                uint32_t* __restrict__ g_out, uint64_t* __restrict__ mask_out, const uint32_t* __restrict__ bin_start,
                uint64_t* __restrict__ lookback, uint32_t* __restrict__ ticket,
                const uint32_t* __restrict__ only_if /* nullptr, or: do nothing when *only_if == 0 */,
                const float4* __restrict__ record /* EXACT (exact tile lists): every mask is refined by P13 */,
                uint32_t tile_end) {
  pdl_launch_dependents();
  pdl_wait();
  extern __shared__ __align__(16) unsigned char smem_raw[];
  BinEmitSmem<BITS>& s = *reinterpret_cast<BinEmitSmem<BITS>*>(smem_raw);
  // lazy lists: the launch that emits the entries behind the first slab runs only if a tile was parked. The
  // tiles are handed out by the ticket, which simply goes on counting from the first launch.
  if (only_if && *only_if == 0u) return;
  do {
    if (!bin_emit_tile<BITS, EXACT>(s, n, Mb, boffsets, chunk_owner, keys, visit, blocks_x, g_out, mask_out, bin_start, lookback,
                                    ticket, record, tile_end))
      return;
    __syncthreads();   // the next tile reuses the shared memory
  } while (tile_end);
}

// ---- 3./4. the walks over a block's entries --------------------------------------------------
constexpr int BW_THREADS = 256;                       // 8 warps = 4 chunks x 2 halves of the block
constexpr int BW_CHUNKS_PER_CTA = BW_THREADS / 64;

// Row `lane` of the transpose of the 32 x 32 bit matrix whose row r is lane r's x.
__device__ __forceinline__ uint32_t transpose32(uint32_t x, uint32_t lane) {
#pragma unroll
  for (int j = 16; j >= 1; j >>= 1) {
    const uint32_t L = j == 16 ? 0x0000FFFFu : j == 8 ? 0x00FF00FFu : j == 4 ? 0x0F0F0F0Fu : j == 2 ? 0x33333333u : 0x55555555u;
    const uint32_t o = __shfl_xor_sync(0xffffffffu, x, j);
    x = (lane & j) ? ((x & ~L) | ((o & ~L) >> j)) : ((x & L) | ((o & L) << j));
  }
  return x;
}

// Which chunk does this warp own? CTAs take tickets so that a chunk only ever waits (look-back)
// on chunks whose CTA has already started. Fills the entry range [e0, e1), the block and whether
// the chunk is the block's first; returns false past the end.
struct BinWalk {
  uint32_t chunk, half, e0, e1, bin, kin, limit;   // kin: index of the chunk inside its block; limit: chunks of the block this round
  bool first;
};
// kin_lo, kin_hi: only the chunks kin_lo <= kin < kin_hi of every block are walked (lazy lists: the first
// kin_hi chunks, later the rest). With kin_lo == 0 and kin_hi < 2^30 the launch enumerates (block, kin) pairs
// directly -- chunk t of the launch is chunk t % kin_hi of block t / kin_hi -- so that its grid is nblocks *
// kin_hi chunks instead of all of them; inside a block kin still ascends with the ticket.
// avail (lazy emission): avail[b] (low 62 bits) = entries of block b that exist so far; a chunk counts only if all
// of its entries do. The first round then stops at min(kin_hi, whole chunks available) per block, and the round
// after it (kin_lo > 0) starts there.
__device__ __forceinline__ uint32_t bin_round0_chunks(const uint32_t* __restrict__ bin_start, const uint64_t* __restrict__ avail,
                                                      uint32_t bin, uint32_t nch, uint32_t c0) {
  uint32_t have = nch;
  if (avail) {
    const uint32_t a = (uint32_t)(avail[bin] & LB_VALUE_MASK), total = bin_start[bin + 1] - bin_start[bin];
    have = a >= total ? nch : a / (uint32_t)BB_CHUNK;
  }
  return min(c0, have);
}

__device__ __forceinline__ bool bin_walk_setup(const uint32_t* __restrict__ bin_start, const uint32_t* __restrict__ chunk_start,
                                               uint32_t* s_cs, uint32_t* __restrict__ ticket, BinWalk& w,
                                               uint32_t kin_lo, uint32_t kin_hi, const uint64_t* __restrict__ avail) {
  if (threadIdx.x == 0) s_cs[BB_MAX_BINS + 1] = atomicAdd(ticket, 1u);
  for (uint32_t k = threadIdx.x; k <= BB_MAX_BINS; k += BW_THREADS) s_cs[k] = chunk_start[k];
  __syncthreads();
  const uint32_t warp = threadIdx.x >> 5;
  const uint32_t t = s_cs[BB_MAX_BINS + 1] * BW_CHUNKS_PER_CTA + (warp >> 1);
  w.half = warp & 1u;
  uint32_t lo;
  if (kin_lo == 0 && kin_hi < (1u << 30)) {
    lo = t / kin_hi;
    w.kin = t - lo * kin_hi;
    if (lo >= BB_MAX_BINS) return false;
    w.limit = bin_round0_chunks(bin_start, avail, lo, s_cs[lo + 1] - s_cs[lo], kin_hi);
    if (w.kin >= w.limit) return false;
    w.chunk = s_cs[lo] + w.kin;
  } else {
    w.chunk = t;
    if (w.chunk >= s_cs[BB_MAX_BINS]) return false;
    lo = 0;
    uint32_t hi = BB_MAX_BINS;   // last b with chunk_start[b] <= chunk: the block that owns it
    while (hi - lo > 1) {
      const uint32_t mid = (lo + hi) >> 1;
      if (s_cs[mid] <= w.chunk) lo = mid; else hi = mid;
    }
    w.kin = w.chunk - s_cs[lo];
    w.limit = kin_hi;
    if (w.kin >= kin_hi) return false;
    if (kin_lo && w.kin < bin_round0_chunks(bin_start, avail, lo, s_cs[lo + 1] - s_cs[lo], kin_lo)) return false;
  }
  w.bin = lo;
  w.first = w.kin == 0;
  w.e0 = bin_start[lo] + w.kin * BB_CHUNK;
  w.e1 = min(w.e0 + (uint32_t)BB_CHUNK, bin_start[lo + 1]);
  return true;
}

// ballot of "bit `bit` of m is set" (test + vote: two instructions)
__device__ __forceinline__ uint32_t ballot_bit(uint32_t m, uint32_t bit) {
  uint32_t w;
  asm volatile("{\n\t"
               ".reg .pred p;\n\t"
               ".reg .b32 t;\n\t"
               "and.b32 t, %1, %2;\n\t"
               "setp.ne.u32 p, t, 0;\n\t"
               "vote.sync.ballot.b32 %0, p, 0xffffffff;\n\t"
               "}"
               : "=r"(w)
               : "r"(m), "r"(bit));
  return w;
}

// The sorted value list. A warp owns (chunk, half of the block's tiles) and holds the whole chunk in
// registers: lane j has entries e0 + 32 b + j, b = 0..15. Tile by tile, the ballot of "my entry covers
// it" ranks the 32 entries of a batch, and the covering lanes store their Gaussian index at consecutive
// positions of that tile's list. The 16 stores of a tile are issued back to back and extend one
// contiguous run (~1 KB), so L2 sees whole lines and DRAM whole bursts.
// s_ptr[l][b]: where batch b's covering entries of tile l go (a pointer into the tile's list), laid down
// by lane l after the look-back. A step is then: test my mask bit, ballot, rank = popcount below my lane,
// address, store -- six instructions plus half a broadcast shared load.
// Measured alternatives (cfg 3, profiles/): a running position advanced by a second popcount per step
// (XU pipe 80% busy), per-batch offsets fetched by shuffles (0.34 ms), the transposed coverage word
// fetched by a shuffle instead of the ballot (0.55 ms: the shuffle path saturates first), compacting each
// tile's run in shared memory and storing whole aligned lines (0.43 ms: more instructions, and the
// partial-line stores were never the limiter -- L2 merges them), the coverage words laid down tile-major in
// shared memory and fetched by broadcast loads instead of the ballots (0.35 ms).
// The pointer rows are padded (BW_PTR_ROW) rather than swizzled: lane l still writes row l without bank
// conflicts, and the loads of the loop are row + constant offset (three address instructions per load
// fewer: 0.325 -> 0.303 ms). With every store confined to an L2-resident window the kernel still takes
// 0.288 ms: it is bound by instruction issue (ALU and XU pipes: LOP3 / VOTE / POPC), not by DRAM.
constexpr int BW_PTR_ROW = BB_CHUNK / 64 + 1;   // uint4 per tile row, padded by one: lane l writes row l without bank conflicts
template <bool FULL>
__device__ __forceinline__ void bin_write_tiles(const uint32_t (&m)[BB_CHUNK / 32], const uint32_t (&g)[BB_CHUNK / 32],
                                                const ulonglong2* s_ptr /* [32 tiles][BW_PTR_ROW] of this warp */, uint32_t nb,
                                                uint32_t lt, uint32_t want /* tiles to write (bit l = tile l) */) {
  for (uint32_t l = 0; l < 32; ++l, s_ptr += BW_PTR_ROW) {
    const uint32_t bit = 1u << l;
    if (!(want & bit)) continue;
#pragma unroll
    for (int k = 0; k < BB_CHUNK / 64; ++k) {
      const ulonglong2 q = s_ptr[k];   // two pointers, broadcast; row + constant offset: no address arithmetic per load
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int b = 2 * k + h;
        if (FULL || b < nb) {
          const uint32_t wl = ballot_bit(m[b], bit);
          uint32_t* dst = reinterpret_cast<uint32_t*>(h ? q.y : q.x);
          if (m[b] & bit) asm volatile("st.global.u32 [%0], %1;" ::"l"(dst + __popc(wl & lt)), "r"(g[b]) : "memory");
        }
      }
    }
  }
}

// ---- exact tile lists (P13): per-tile and per-Gaussian counts of the refined masks, then the ranges ----------------
// With refined masks a tile's count is no longer the number of rectangles over it (tilebin.cuh's difference array):
// it is counted. A warp owns (chunk, half of the block's tiles) exactly as in bin_write_kernel below: the counts per tile
// come from the bit-matrix transpose + popcount, one atomicAdd per (chunk, tile); each lane also adds its entries'
// popcounts to its Gaussians' exact counts. Integer adds commute: deterministic.
__global__ void __launch_bounds__(BW_THREADS, 4)
exact_count_kernel(const uint32_t* __restrict__ gs, const uint64_t* __restrict__ masks, const uint32_t* __restrict__ bin_start,
                   const uint32_t* __restrict__ chunk_start, uint32_t tiles_x, uint32_t tiles_y, uint32_t blocks_x,
                   uint32_t* __restrict__ ticket, uint32_t* __restrict__ tile_count /* [tiles], zeroed */,
                   uint32_t* __restrict__ gauss_count /* [n], zeroed */) {
  __shared__ uint32_t s_cs[BB_MAX_BINS + 2];
  BinWalk w;
  if (!bin_walk_setup(bin_start, chunk_start, s_cs, ticket, w, 0u, 0xFFFFFFFFu, nullptr)) return;
  const uint32_t lane = threadIdx.x & 31u;
  constexpr int NB = BB_CHUNK / 32;
  const uint32_t* mp = reinterpret_cast<const uint32_t*>(masks) + w.half;   // this half's 32 mask bits
  uint32_t cnt = 0;
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    const uint32_t e = w.e0 + b * 32 + lane;
    const bool ok = e < w.e1;
    const uint32_t m = ok ? __ldcs(mp + 2 * (size_t)e) : 0u;
    if (m) atomicAdd(gauss_count + __ldcs(gs + e), (uint32_t)__popc(m));
    cnt += __popc(transpose32(m, lane));
  }
  const uint32_t ltile = w.half * 32u + lane;
  const uint32_t tx = (w.bin % blocks_x) * 8u + (ltile & 7u), ty = (w.bin / blocks_x) * 8u + (ltile >> 3);
  if (cnt && tx < tiles_x && ty < tiles_y) atomicAdd(tile_count + ty * tiles_x + tx, cnt);
}

// ranges[tile] = exclusive scan of the exact counts in row-major tile order; one CTA. total -> totals[0] (device) and
// totals_host[7] (mapped).
__global__ void __launch_bounds__(1024)
exact_ranges_kernel(const uint32_t* __restrict__ tile_count, uint32_t tiles, uint2* __restrict__ ranges,
                    uint64_t* __restrict__ total_dev, volatile uint64_t* __restrict__ totals_host) {
  __shared__ uint64_t s_part[32];
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t per = (tiles + 1023u) / 1024u;
  const uint32_t t0 = min(tiles, tid * per), t1 = min(tiles, t0 + per);
  uint64_t sum = 0;
  for (uint32_t t = t0; t < t1; ++t) sum += tile_count[t];
  uint64_t incl = sum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint64_t v = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= d) incl += v;
  }
  if (lane == 31) s_part[warp] = incl;
  __syncthreads();
  uint64_t wex = 0, all = 0;
  for (uint32_t wv = 0; wv < 32; ++wv) {
    const uint64_t v = s_part[wv];
    if (wv < warp) wex += v;
    all += v;
  }
  uint64_t run = wex + incl - sum;
  for (uint32_t t = t0; t < t1; ++t) {
    const uint32_t c = tile_count[t];
    ranges[t] = make_uint2((uint32_t)run, (uint32_t)(run + c));
    run += c;
  }
  if (tid == 0) { *total_dev = all; totals_host[7] = all; }
}

// status[chunk][64]: 64-bit look-back words (flag | position), zeroed. A chunk first counts, per tile,
// how many of its entries cover it (bit-matrix transpose + popcount), publishes the counts, resolves
// where it starts in every tile list by looking back over the earlier chunks of its block (the block's
// first chunk starts at the tile's range begin), and then writes.
// One ticket's BW_CHUNKS_PER_CTA chunks. *past_end (block-uniform): the ticket lies beyond the launch's last chunk.
__device__ __forceinline__ void
bin_write_ticket(uint32_t* s_cs, uint32_t* const* s_vals, ulonglong2 (*s_ptr)[32 * BW_PTR_ROW], bool* past_end,
                 const uint32_t* __restrict__ gs, const uint64_t* __restrict__ masks, const uint32_t* __restrict__ bin_start,
                 const uint32_t* __restrict__ chunk_start, const uint2* __restrict__ ranges, uint32_t tiles_x,
                 uint32_t tiles_y, uint32_t blocks_x, uint64_t* __restrict__ status, uint32_t* __restrict__ ticket,
                 uint32_t kin_lo, uint32_t kin_hi, const unsigned long long* __restrict__ want_mask, uint32_t* __restrict__ lim,
                 const uint64_t* __restrict__ avail) {
  BinWalk w;
  const bool mine = bin_walk_setup(bin_start, chunk_start, s_cs, ticket, w, kin_lo, kin_hi, avail);   // (contains the barrier)
  {
    const uint32_t first = s_cs[BB_MAX_BINS + 1] * BW_CHUNKS_PER_CTA;
    *past_end = (kin_lo == 0 && kin_hi < (1u << 30)) ? first / kin_hi >= (uint32_t)BB_MAX_BINS : first >= s_cs[BB_MAX_BINS];
  }
  if (!mine) return;
  // lazy lists, second round: only the tiles the blend has not finished; a block without any is skipped by all of
  // its chunks alike (the mask is fixed for the whole launch), so nobody waits for a skipped chunk's look-back word
  const uint32_t want = want_mask ? (uint32_t)(want_mask[w.bin] >> (32u * w.half)) : 0xFFFFFFFFu;
  if (want_mask && want_mask[w.bin] == 0ull) return;
  uint32_t* const vp = *s_vals;
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t lt = lanemask_lt();
  constexpr int NB = BB_CHUNK / 32;
  const uint32_t* mp = reinterpret_cast<const uint32_t*>(masks) + w.half;   // this half's 32 mask bits
  uint32_t m[NB], g[NB];
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    const uint32_t e = w.e0 + b * 32 + lane;
    const bool ok = e < w.e1;
    m[b] = ok ? __ldcs(mp + 2 * (size_t)e) : 0u;
    g[b] = ok ? __ldcs(gs + e) : 0u;
  }
  // lane = tile (half * 32 + lane) of the block from here to the end of the look-back
  uint32_t cnt = 0;
  uint32_t pre[NB];   // covering entries of my tile in the batches before batch b
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    pre[b] = cnt;
    cnt += __popc(transpose32(m[b], lane));
  }
  uint64_t* my = status + (size_t)w.chunk * 64u + w.half * 32u + lane;
  uint32_t mypos;
  if (w.first) {
    const uint32_t ltile = w.half * 32u + lane;
    const uint32_t tx = (w.bin % blocks_x) * 8u + (ltile & 7u), ty = (w.bin / blocks_x) * 8u + (ltile >> 3);
    mypos = (tx < tiles_x && ty < tiles_y) ? ranges[ty * tiles_x + tx].x : 0u;
  } else {
    st_relaxed_u64(my, LB_FLAG_AGG | cnt);
    mypos = 0;
    // windowed look-back: the status words of the next LB_WINDOW predecessors are fetched together (the
    // chunks of a wave start at the same time, so their prefixes lag and the walk can be long), then
    // consumed in order up to the first one that is not published yet
#ifndef PVG_BW_LB_WINDOW
#define PVG_BW_LB_WINDOW 4
#endif
    constexpr int LB_WINDOW = PVG_BW_LB_WINDOW;
    const uint64_t* p = my - 64;
    uint32_t left = w.kin;   // predecessors inside the block; the block's first chunk always ends the walk
    bool done = false;
    while (!done) {
      uint64_t v[LB_WINDOW];
#pragma unroll
      for (int k = 0; k < LB_WINDOW; ++k) v[k] = (uint32_t)k < left ? ld_relaxed_u64(p - 64 * k) : 0ull;
      uint32_t used = 0;
      bool open = true;
#pragma unroll
      for (int k = 0; k < LB_WINDOW; ++k) {
        const uint64_t flag = v[k] & LB_FLAG_MASK;
        open = open && flag != 0;   // a zero flag: that chunk's CTA holds an earlier ticket, it is running
        if (open) {
          mypos += (uint32_t)v[k];
          ++used;
          if (flag == LB_FLAG_PREFIX) { done = true; open = false; }
        }
      }
      p -= 64 * used;
      left -= used;
    }
  }
  st_relaxed_u64(my, LB_FLAG_PREFIX | (uint64_t)(mypos + cnt));
  if (lim && w.kin + 1u == w.limit) {
    // the last chunk of the block this round writes: the blend's first phase reads each list up to here
    const uint32_t ltile = w.half * 32u + lane;
    const uint32_t tx = (w.bin % blocks_x) * 8u + (ltile & 7u), ty = (w.bin / blocks_x) * 8u + (ltile >> 3);
    if (tx < tiles_x && ty < tiles_y) lim[ty * tiles_x + tx] = mypos + cnt;
  }
  ulonglong2* sp = s_ptr[threadIdx.x >> 5];
  {
    const uint64_t base = reinterpret_cast<uint64_t>(vp + mypos);
#pragma unroll
    for (int k = 0; k < NB / 2; ++k) {
      const uint64_t a = base + 4ull * pre[2 * k], c = base + 4ull * pre[2 * k + 1];
      sp[BW_PTR_ROW * lane + k] = make_ulonglong2(a, c);
    }
  }
  __syncwarp();
  const uint32_t nb = (w.e1 - w.e0 + 31u) >> 5;
  if (nb == NB) bin_write_tiles<true>(m, g, sp, nb, lt, want);
  else bin_write_tiles<false>(m, g, sp, nb, lt, want);
}

// loop == 0: one ticket per CTA (the grid covers the launch's chunks). loop != 0: the CTAs loop over tickets to the
// launch's last chunk -- the second round of the lazy lists, which usually finds nothing to do (*want_count == 0) and
// should then cost a few hundred CTAs. Tickets are taken in order by running CTAs, so a chunk still only ever waits
// (look-back) on chunks that are done or being worked on.
__global__ void __launch_bounds__(BW_THREADS, 4)
bin_write_kernel(const uint32_t* __restrict__ gs, const uint64_t* __restrict__ masks, const uint32_t* __restrict__ bin_start,
                 const uint32_t* __restrict__ chunk_start, const uint2* __restrict__ ranges, uint32_t tiles_x,
                 uint32_t tiles_y, uint32_t blocks_x, uint64_t* __restrict__ status, uint32_t* __restrict__ ticket,
                 uint32_t* __restrict__ vals, uint32_t kin_lo, uint32_t kin_hi,
                 const unsigned long long* __restrict__ want_mask /* [blocks] tiles still wanted, or nullptr: all */,
                 const uint32_t* __restrict__ want_count /* with want_mask: nothing to do at all if 0 */,
                 uint32_t* __restrict__ lim /* [tiles] or nullptr: where each tile's list stands after this round */,
                 const uint64_t* __restrict__ avail /* [blocks] or nullptr: entries emitted so far (bin_round0_chunks) */,
                 uint32_t loop) {
  pdl_launch_dependents();
  pdl_wait();
  __shared__ uint32_t s_cs[BB_MAX_BINS + 2];
  // the base pointer round-trips through shared memory so that it lives in registers; taken from the
  // kernel parameter it is re-read from the constant bank before every store (one more instruction per step)
  __shared__ uint32_t* s_vals;
  __shared__ ulonglong2 s_ptr[BW_THREADS / 32][32 * BW_PTR_ROW];
  if (want_mask && *want_count == 0u) return;   // lazy lists: no tile was parked
  if (threadIdx.x == 0) s_vals = vals;
  do {
    bool past_end;
    bin_write_ticket(s_cs, &s_vals, s_ptr, &past_end, gs, masks, bin_start, chunk_start, ranges, tiles_x, tiles_y, blocks_x, status,
                     ticket, kin_lo, kin_hi, want_mask, lim, avail);
    if (past_end) return;   // block-uniform
    __syncthreads();        // the next ticket's setup rewrites s_cs
  } while (loop);
}

}  // namespace pvg

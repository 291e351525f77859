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
constexpr int OS_MAX_PASSES = 10;

struct SortPlan {
  int num_passes;
  int shift[OS_MAX_PASSES];
  int bits[OS_MAX_PASSES];
};

// Split [begin_bit, end_bit) into digit passes of at most 8 bits and near-equal width
// (14 -> 7+7). No pass straddles bit 32, so a digit always comes from one 32-bit half.
inline SortPlan make_sort_plan(int begin_bit, int end_bit) {
  SortPlan p{};
  auto seg = [&](int b0, int b1) {
    const int B = b1 - b0;
    if (B <= 0) return;
    const int np = (B + OS_RADIX_BITS - 1) / OS_RADIX_BITS;
    int at = b0;
    for (int i = 0; i < np; ++i) {
      const int left = b1 - at, passes_left = np - i;
      const int b = (left + passes_left - 1) / passes_left;
      p.shift[p.num_passes] = at;
      p.bits[p.num_passes] = b;
      ++p.num_passes;
      at += b;
    }
  };
  seg(begin_bit, end_bit < 32 ? end_bit : (begin_bit < 32 ? 32 : begin_bit));
  seg(begin_bit > 32 ? begin_bit : 32, end_bit);
  return p;
}

// Lanes of the warp holding the same digit as the caller: one vote.ballot per digit bit.
// On sm_100a MATCH.ANY runs on the address-divergence unit at ~64 cycles per warp
// instruction per SM and capped a sort pass near 40% of HBM bandwidth (profiles/), while
// ballots issue on the regular pipes.
template <int BITS>
__device__ __forceinline__ uint32_t digit_peers(uint32_t d) {
  uint32_t peers = 0xffffffffu;
#pragma unroll
  for (int b = 0; b < BITS; ++b) {
    // 4 instructions per bit: test (LOP3 with predicate out), ballot, select, and-xor
    asm("{\n\t"
        ".reg .pred p;\n\t"
        ".reg .b32 t, m, x;\n\t"
        "and.b32 t, %1, %2;\n\t"
        "setp.ne.u32 p, t, 0;\n\t"
        "vote.sync.ballot.b32 m, p, 0xffffffff;\n\t"
        "selp.b32 x, 0, -1, p;\n\t"
        "lop3.b32 %0, %0, m, x, 0x60;\n\t"   // peers & (m ^ x)
        "}"
        : "+r"(peers)
        : "r"(d), "r"(1u << b));
  }
  return peers;
}

// ---- digit histograms of every pass in one read of the keys ---------------------------
constexpr int HIST_THREADS = 512;
constexpr int HIST_ITEMS = 8;

// AGGREGATE: equal digits inside a warp are combined before the shared-memory atomic -- right for the
// tile-id digits of an instance list (neighbours nearly always agree), wasteful for depth bits (the
// eight ballots per digit cost more than the plain atomics: 0.045 ms against 0.0xx ms on 3M keys).
template <bool AGGREGATE>
__global__ void __launch_bounds__(HIST_THREADS)
onesweep_histogram_kernel(const uint64_t* __restrict__ keys, uint64_t n, const __grid_constant__ SortPlan plan,
                          uint32_t* __restrict__ hist /* [passes][256]: counts, then exclusive prefixes */,
                          uint32_t* __restrict__ done /* zeroed: CTAs that have added their counts */) {
  __shared__ uint32_t s_hist[OS_MAX_PASSES * OS_RADIX];
  for (int k = threadIdx.x; k < plan.num_passes * OS_RADIX; k += HIST_THREADS) s_hist[k] = 0;
  __syncthreads();
  // block-uniform trip count
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
      const uint32_t live = AGGREGATE ? __ballot_sync(0xffffffffu, ok) : 0u;
      for (int p = 0; p < plan.num_passes; ++p) {
        const uint32_t d = (uint32_t)(k[u] >> plan.shift[p]) & ((1u << plan.bits[p]) - 1u);
        if (AGGREGATE) {
          const uint32_t peers = digit_peers<OS_RADIX_BITS>(d) & live;
          if (ok && (peers & lt) == 0) atomicAdd(&s_hist[p * OS_RADIX + d], (uint32_t)__popc(peers));
        } else if (ok) {
          atomicAdd(&s_hist[p * OS_RADIX + d], 1u);
        }
      }
    }
  }
  __syncthreads();
  for (int k = threadIdx.x; k < plan.num_passes * OS_RADIX; k += HIST_THREADS) {
    const uint32_t v = s_hist[k];
    if (v) atomicAdd(&hist[k], v);
  }
  // the last CTA to arrive turns the counts into exclusive prefixes (saves a launch: the scan is 1 KB per pass)
  __shared__ bool s_last;
  __shared__ uint32_t s_warp[OS_RADIX / 32];
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) s_last = atomicAdd(done, 1u) == gridDim.x - 1;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
  for (int p = 0; p < plan.num_passes; ++p) {
    uint32_t v = 0, incl = 0;
    if (threadIdx.x < OS_RADIX) {
      v = __ldcg(hist + p * OS_RADIX + threadIdx.x);
      incl = v;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += t;
      }
      if (lane == 31) s_warp[warp] = incl;
    }
    __syncthreads();
    if (threadIdx.x < OS_RADIX) {
      uint32_t wex = 0;
      for (uint32_t w = 0; w < warp; ++w) wex += s_warp[w];
      hist[p * OS_RADIX + threadIdx.x] = wex + incl - v;
    }
    __syncthreads();
  }
}

// ---- the ranking core shared by every digit pass ----------------------------------------
// A tile of THREADS*ITEMS elements is held warp-striped: warp w owns ITEMS*32 consecutive
// elements, lane l its elements l, l+32, ... (so a "row" j of a warp is 32 consecutive
// elements). rank() turns the per-element digits into tile-local sorted positions and
// resolves, by decoupled look-back over earlier tiles, where each digit's run starts in the
// output. Stable: earlier rows, lower lanes, lower warps, earlier tiles come first.
#ifndef PVG_LB_WINDOW
#define PVG_LB_WINDOW 4
#endif
template <int THREADS, int ITEMS, int BITS>
struct RadixCore {
  static constexpr int WARPS = THREADS / 32;
  static constexpr int TILE = THREADS * ITEMS;
  static constexpr int RADIX = 1 << BITS;
  static constexpr int DWARPS = (RADIX + 31) / 32;  // warps that hold the digit threads
  static constexpr int DSHIFT = BITS <= 8 ? 8 : BITS;   // dp = digit | position << DSHIFT
  static constexpr uint32_t DMASK = (1u << DSHIFT) - 1u;
  static constexpr uint32_t INVALID = 0xFFFFFFFFu;      // SPARSE: "no element here"
  static_assert(THREADS >= RADIX && TILE < 65536 && DSHIFT + 16 <= 32, "digit threads / u16 positions");

  struct Smem {
    uint32_t warp_off[WARPS * RADIX];  // per-warp digit counts -> tile-local start of (warp, digit)
    uint32_t out_base[RADIX];          // output index of the digit's run MINUS its tile-local start
    uint32_t warp_sums[DWARPS];
    uint32_t tile;
    uint32_t total;                    // elements of the tile that take part (SPARSE: the valid ones)
  };

  __device__ static __forceinline__ uint32_t take_ticket(Smem& s, uint32_t* ticket) {
    if (threadIdx.x == 0) s.tile = atomicAdd(ticket, 1u);
    for (int k = threadIdx.x; k < WARPS * RADIX; k += THREADS) s.warp_off[k] = 0;
    __syncthreads();
    return s.tile;
  }

  // In: dp[j] = digit of the thread's j-th element (padding elements carry RADIX-1 and must
  // be the last elements of the tile). Out: dp[j] = digit | tile-local sorted position << DSHIFT
  // (packed to save registers). Ends with a __syncthreads(); afterwards
  // s.out_base[digit] + position is the element's output index.
  // SPARSE: elements with dp[j] == INVALID take no part (anywhere in the tile): they are not counted, get no
  // position and keep dp[j] == INVALID; s.total is the number of elements that do take part.
  // WINDOW: look-back words fetched per round trip. Large sorts run in waves and find a published prefix nearby (4 is
  // enough); a small sort's tiles all start together, and a tile walks back over all of them.
  template <bool SPARSE = false, int WINDOW = PVG_LB_WINDOW>
  __device__ static __forceinline__ void rank(Smem& s, uint32_t tile, uint32_t (&dp)[ITEMS],
                                              const uint32_t* __restrict__ hist_excl,
                                              uint64_t* __restrict__ lookback) {
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    uint32_t* wh = s.warp_off + warp * RADIX;
    const uint32_t lt = lanemask_lt();
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const bool ok = !SPARSE || dp[j] != INVALID;
      const uint32_t d = ok ? dp[j] : 0u;
      uint32_t peers = digit_peers<BITS>(d);
      if (SPARSE) peers &= __ballot_sync(0xffffffffu, ok);
      const uint32_t before = wh[d];
      __syncwarp();
      if (ok && (peers & lt) == 0) wh[d] = before + __popc(peers);
      __syncwarp();
      dp[j] = ok ? (d | ((before + __popc(peers & lt)) << DSHIFT)) : INVALID;
    }
    __syncthreads();

    if (tid < DWARPS * 32) {  // whole warps, so the shuffles and the named barrier are uniform
      const bool live = tid < RADIX;
      // digit thread: exclusive scan of the warp counts over warps -> the tile's digit count
      uint32_t tile_count = 0;
      if (live) {
#pragma unroll
        for (int w = 0; w < WARPS; ++w) tile_count += s.warp_off[w * RADIX + tid];
      }
      // publish this tile's digit count before anything else: later tiles look back at it
      uint64_t* my = lookback + (uint64_t)tile * RADIX + tid;
      if (live) st_relaxed_u64(my, (tile == 0 ? LB_FLAG_PREFIX : LB_FLAG_AGG) | tile_count);
      // exclusive scan of the tile counts over digits -> tile-local bin starts
      uint32_t incl = tile_count;
#pragma unroll
      for (int k = 1; k < 32; k <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, k);
        if (lane >= k) incl += t;
      }
      if (lane == 31) s.warp_sums[warp] = incl;
      asm volatile("bar.sync 1, %0;" ::"n"(DWARPS * 32));
      uint32_t start = incl - tile_count;
#pragma unroll
      for (int w = 0; w < DWARPS; ++w)
        if (w < (int)warp) start += s.warp_sums[w];
      if (tid == RADIX - 1) s.total = start + tile_count;
      if (live) {
        uint32_t run = start;
#pragma unroll
        for (int w = 0; w < WARPS; ++w) {
          const uint32_t c = s.warp_off[w * RADIX + tid];
          s.warp_off[w * RADIX + tid] = run;
          run += c;
        }
        // resolve the exclusive prefix of this digit over earlier tiles
        uint32_t excl = 0;
        if (tile != 0) {
          // windowed: the status words of the next LB_WINDOW predecessors are fetched together (one L2
          // round trip), then consumed in order up to the first one that is not published yet
          constexpr int LB_WINDOW = WINDOW;
          uint32_t left = tile;   // predecessors not yet consumed; tile 0 always ends the walk
          const uint64_t* p = lookback + (uint64_t)(tile - 1) * RADIX + tid;
          bool done = false;
          while (!done) {
            uint64_t v[LB_WINDOW];
#pragma unroll
            for (int k = 0; k < LB_WINDOW; ++k) v[k] = (uint32_t)k < left ? ld_relaxed_u64(p - (size_t)k * RADIX) : 0ull;
            uint32_t used = 0;
            bool open = true;
#pragma unroll
            for (int k = 0; k < LB_WINDOW; ++k) {
              const uint64_t flag = v[k] & LB_FLAG_MASK;
              open = open && flag != 0;   // zero: that tile holds an earlier ticket, it is running
              if (open) {
                excl += (uint32_t)v[k];
                ++used;
                if (flag == LB_FLAG_PREFIX) { done = true; open = false; }
              }
            }
            p -= (size_t)used * RADIX;
            left -= used;
          }
          st_relaxed_u64(my, LB_FLAG_PREFIX | (uint64_t)(uint32_t)(excl + tile_count));
        }
        s.out_base[tid] = hist_excl[tid] + excl - start;  // mod 2^32 (n < 2^32)
      }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < ITEMS; ++j)
      if (!SPARSE || dp[j] != INVALID) dp[j] += wh[dp[j] & DMASK] << DSHIFT;
  }
};

// ---- one digit pass over (u64 key, u32 value) pairs --------------------------------------
template <int THREADS, int ITEMS, int BITS>
struct OnesweepSmem {
  typename RadixCore<THREADS, ITEMS, BITS>::Smem core;
  uint64_t keys[THREADS * ITEMS];
  uint32_t vals[THREADS * ITEMS];
};

// The digit is bits [shift32, shift32+BITS) of the key's upper (HI = 1) or lower 32-bit
// half (make_sort_plan never lets a pass straddle bit 32). Elements are re-ordered through
// shared memory and written out in digit runs so that stores are coalesced.
// STREAM: read the pairs with evict-first loads (lists far larger than L2); otherwise leave them in L2
// for the next pass (the n-key depth sort: 36 MB at 3M Gaussians).
template <int THREADS, int ITEMS, int BITS, int MINB, int HI, bool STREAM>
__global__ void __launch_bounds__(THREADS, MINB)
onesweep_pass_kernel(const uint64_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                     uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out, uint32_t n,
                     int shift32, const uint32_t* __restrict__ hist_excl /* [256] this pass */,
                     uint64_t* __restrict__ lookback /* [tiles][1 << BITS], zeroed */,
                     uint32_t* __restrict__ ticket /* zeroed */) {
  using Core = RadixCore<THREADS, ITEMS, BITS>;
  constexpr int TILE = Core::TILE;
  constexpr uint32_t MASK = (1u << BITS) - 1u;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  OnesweepSmem<THREADS, ITEMS, BITS>& s = *reinterpret_cast<OnesweepSmem<THREADS, ITEMS, BITS>*>(smem_raw);

  const uint32_t tile = Core::take_ticket(s.core, ticket);
  const uint32_t tile_base = tile * TILE;
  const uint32_t tile_n = min((uint32_t)TILE, n - tile_base);
  const uint32_t tid = threadIdx.x;
  const uint32_t wbase = (tid >> 5) * (ITEMS * 32) + (tid & 31u);

  // load (warp-striped); padding keys are all-ones: they rank after every real key of the
  // last digit and are never written
  const uint64_t* kp = keys_in + tile_base + wbase;
  const uint32_t* vp = vals_in + tile_base + wbase;
  uint64_t key[ITEMS];
  uint32_t val[ITEMS];
  if (tile_n == TILE) {
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) key[j] = STREAM ? __ldcs(kp + j * 32) : __ldcg(kp + j * 32);
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) val[j] = STREAM ? __ldcs(vp + j * 32) : __ldcg(vp + j * 32);
  } else {
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const bool ok = wbase + j * 32 < tile_n;
      key[j] = ok ? (STREAM ? __ldcs(kp + j * 32) : __ldcg(kp + j * 32)) : ~0ull;
      val[j] = ok ? (STREAM ? __ldcs(vp + j * 32) : __ldcg(vp + j * 32)) : 0u;
    }
  }
  uint32_t dp[ITEMS];
#pragma unroll
  for (int j = 0; j < ITEMS; ++j) {
    const uint32_t w = HI ? (uint32_t)(key[j] >> 32) : (uint32_t)key[j];
    dp[j] = (w >> shift32) & MASK;
  }
  Core::rank(s.core, tile, dp, hist_excl, lookback);

#pragma unroll
  for (int j = 0; j < ITEMS; ++j) {
    s.keys[dp[j] >> Core::DSHIFT] = key[j];
    s.vals[dp[j] >> Core::DSHIFT] = val[j];
  }
  __syncthreads();

  // coalesced write-out of digit runs (real keys occupy local positions [0, tile_n))
  for (uint32_t p = tid; p < tile_n; p += THREADS) {
    const uint64_t k = s.keys[p];
    const uint32_t w = HI ? (uint32_t)(k >> 32) : (uint32_t)k;
    const uint32_t o = s.core.out_base[(w >> shift32) & MASK] + p;
    keys_out[o] = k;
    vals_out[o] = s.vals[p];
  }
}

// ---- the depth sort of the Gaussians: its own plan and pass kernel ------------------------------
// Keys are the n depth pairs preprocess writes: low half = fp32 bits of z MINUS the fp32 bits of znear (z > znear > 0,
// so the difference is positive and order-preserving; for z up to 65536 znear it is below 2^27), or 0xFFFFFFFF for a
// culled Gaussian; upper half = the packed tile rectangle (payload). 31 key bits in digits of 9 + 9 + 9 + 4:
//   * pass 0 reads all n pairs and DROPS the culled ones (they take no part in its ranking, RadixCore SPARSE), so the
//     later passes, the scan and the list building see the S survivors only (75 % of n at config 3);
//   * a pass whose digit is the same for every key is the identity and exits at once -- the 4-bit top digit of any
//     scene whose far plane is below 65536 znear: three passes instead of the four of an 8-bit plan;
//   * S, which passes run and which buffer each reads are decided on the device by the last CTA of preprocess, which
//     holds the digit histograms (DepthCtl); every pass is launched for the worst case and reads the block.
#ifndef PVG_DS_THREADS
#define PVG_DS_THREADS 512   // tile shape of the depth passes (the launch configuration lives in pvg_api.cu: DsCfg)
#define PVG_DS_ITEMS 8
#define PVG_DS_MINB 2
#endif
constexpr int DS_PASSES = 4;
constexpr int DS_BITS = 9;
constexpr int DS_RADIX = 1 << DS_BITS;
constexpr int DS_TOP_BITS = 31 - 3 * DS_BITS;   // 4
__host__ __device__ constexpr int ds_shift(int p) { return p * DS_BITS; }
__host__ __device__ constexpr int ds_bits(int p) { return p < 3 ? DS_BITS : DS_TOP_BITS; }

// control block in device memory, written by preprocess's last CTA (preprocess.cuh)
struct DepthCtl {
  uint32_t survivors;          // S
  uint32_t final_side;         // which buffer pair holds the sorted pairs
  uint32_t skip[DS_PASSES];    // 1: the pass is the identity
  uint32_t in_side[DS_PASSES]; // buffer pair the pass reads (it writes the other one)
};

// Layout of a histogram region (u32 words) of the depth sort: [4][512] digit counts, turned into exclusive prefixes by
// the last CTA of the kernel that counts them, a CTA counter, the control block.
constexpr int DH_COUNTER = DS_PASSES * DS_RADIX;   // u32 index of the CTA counter (the two words after it: a 64-bit sum)
constexpr int DH_CTL = DH_COUNTER + 8;             // u32 index of the control block (8-byte aligned)
constexpr int DH_WORDS = DH_CTL + 16;              // words per region (a multiple of 4)
static_assert(sizeof(DepthCtl) <= 16 * 4, "DepthCtl fits its slot");

// ---- front-first depth order (lazy lists) -------------------------------------------------------------------------
// The first round of the lazy lists consumes the first slab of the block entries in depth order, and those belong to
// the few Gaussians nearest the camera (they are the large ones: about 1 % of the survivors own the first eighth of
// the entries at config 3). So the frame orders only those: preprocess's last CTA picks a key threshold from a
// histogram of the entries over the top key bits (FrontCtl), depth_select_kernel<false> compacts the pairs below it
// (index order: the sort stays stable) and counts their digits, and the ordinary passes run over that front alone.
// The pairs at and beyond the threshold are selected and ordered behind the front -- a sorted front followed by a sorted
// back IS the sorted whole, the threshold being a key value -- only if a tile parks (second round) or a debug view asks.
constexpr int FR_SHIFT = 18;                       // bucket = key >> 18: 32 buckets per binade of z
constexpr int FR_BUCKETS = 1024;                   // the last one takes every key beyond 1023 << 18
constexpr int FR_TOP = 1 << (3 * DS_BITS - FR_SHIFT);   // buckets below it hold keys below 2^27: top digit 0
struct FrontCtl {
  uint32_t survivors;   // S
  uint32_t front;       // F: pairs with key < thr
  uint32_t thr;         // 0xFFFFFFFF: every survivor is in front
  uint32_t top_front;   // 1: the front has keys of 2^27 and beyond (its top-digit pass is needed)
  uint32_t top_back;    // 1: the back has
};

// One wave: 1024 threads x 24 pairs = 24576 pairs per CTA, 123 CTAs for 3 M pairs. A pass like this is a chain of
// latencies (ticket, loads, look-back, writes, last-CTA count) -- with tiles of 4096 it ran in three waves and took
// three chains (ncu: 36 us, warps waiting at barriers).
#ifndef PVG_SEL_THREADS
#define PVG_SEL_THREADS 1024
#define PVG_SEL_ITEMS 24
#endif
constexpr int SEL_THREADS = PVG_SEL_THREADS;
constexpr int SEL_ITEMS = PVG_SEL_ITEMS;
constexpr int SEL_TILE = SEL_THREADS * SEL_ITEMS;

// Ordered selection of one class of pairs. keys: the n pairs of preprocess in index order (never overwritten).
// Output: the selected pairs (key, index) in index order at keys_out / vals_out [base, base + count), base = 0 (front)
// or F (back), the indices once more in list_out (optional: shade_list_kernel reads them while the passes already
// overwrite vals_out); region: the class's histogram region (zeroed): digit prefixes + DepthCtl for the passes, which
// read buffer `out_side` first. status [tiles] and ticket: zeroed. only_if: nothing to do when *only_if == 0.
// The kernel also zeroes the look-back words its class's passes will use (lb: [4 passes][lb_rows][radix], tiles of
// lb_tile pairs): the class's size is known here (FrontCtl), so no memset sized by n is needed.
// A warp owns 32 x 24 consecutive pairs, element (j, lane) at j * 32 + lane: coalesced loads, and the rank of a
// selected element inside the warp's run is popc of the ballots before it. Only the ballots stay in registers; the
// selected keys are loaded again (few of them in front; all of them, coalesced, behind).
template <bool BACK>
__global__ void __launch_bounds__(SEL_THREADS)
depth_select_kernel(const uint64_t* __restrict__ keys, uint32_t n, const FrontCtl* __restrict__ fc,
                    uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out, uint32_t* __restrict__ list_out,
                    uint32_t* __restrict__ region, uint64_t* __restrict__ status, uint32_t* __restrict__ ticket,
                    uint32_t out_side, uint64_t* __restrict__ lb, uint32_t lb_rows, uint32_t lb_tile,
                    const uint32_t* __restrict__ only_if) {
  pdl_launch_dependents();
  pdl_wait();
  if (only_if && *only_if == 0u) return;
  __shared__ uint32_t s_hist[DS_PASSES * DS_RADIX];
  __shared__ uint32_t s_tile, s_warp[SEL_THREADS / 32], s_first[SEL_THREADS / 32];
  __shared__ uint64_t s_sum[SEL_THREADS / 32];
  __shared__ bool s_last;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
#pragma unroll
  for (int k = 0; k < DS_PASSES * DS_RADIX / SEL_THREADS; ++k) s_hist[k * SEL_THREADS + tid] = 0;
  if (tid == 0) s_tile = atomicAdd(ticket, 1u);
  const uint32_t thr = fc->thr;
  const uint32_t out0 = BACK ? fc->front : 0u;
  {
    const uint32_t cnt = BACK ? fc->survivors - fc->front : fc->front;
    const uint32_t rows = min(lb_rows, (cnt + lb_tile - 1u) / lb_tile);
    uint64_t* q = lb;
    for (int d = 0; d < DS_PASSES; ++d) {
      const uint32_t words = rows << ds_bits(d);
      for (uint32_t i = blockIdx.x * SEL_THREADS + tid; i < words; i += gridDim.x * SEL_THREADS) q[i] = 0ull;
      q += (size_t)lb_rows << ds_bits(d);
    }
  }
  __syncthreads();
  const uint32_t tile = s_tile;
  const uint32_t wbase = tile * SEL_TILE + warp * (32 * SEL_ITEMS) + lane;
  const uint32_t* lo32 = reinterpret_cast<const uint32_t*>(keys);   // the depth key: the low word of the pair
  uint32_t bal[SEL_ITEMS];
  uint32_t wcount = 0;
  constexpr int HALF = SEL_ITEMS / 2;   // the loads of a half are all in flight before the first ballot
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t w[HALF];
#pragma unroll
    for (int j = 0; j < HALF; ++j) {
      const uint32_t i = wbase + (h * HALF + j) * 32;
      w[j] = i < n ? __ldcg(lo32 + 2 * (size_t)i) : 0xFFFFFFFFu;
    }
#pragma unroll
    for (int j = 0; j < HALF; ++j) {
      const bool in = BACK ? (w[j] >= thr && w[j] != 0xFFFFFFFFu) : (w[j] < thr);
      bal[h * HALF + j] = __ballot_sync(0xffffffffu, in);
      wcount += __popc(bal[h * HALF + j]);
    }
  }
  if (lane == 0) s_warp[warp] = wcount;
  __syncthreads();
  uint32_t warp_excl = 0, block_sum = 0;
#pragma unroll
  for (int w = 0; w < SEL_THREADS / 32; ++w) {
    const uint32_t v = s_warp[w];
    if (w < (int)warp) warp_excl += v;
    block_sum += v;
  }
  // Look-back over the tiles' counts, the whole CTA wide: thread t waits for the word of tile - 1 - t (it holds an
  // earlier ticket: its CTA is running), the CTA adds the counts up to the nearest published prefix.
  uint64_t excl = 0;
  if (tile == 0) {
    if (tid == 0) st_relaxed_u64(status, LB_FLAG_PREFIX | block_sum);
  } else {
    if (tid == 0) st_relaxed_u64(status + tile, LB_FLAG_AGG | block_sum);
    int64_t p = (int64_t)tile - 1 - (int64_t)tid;
    while (true) {
      uint64_t sv = LB_FLAG_PREFIX;
      if (p >= 0) do { sv = ld_relaxed_u64(status + p); } while ((sv & LB_FLAG_MASK) == 0ull);
      const uint32_t pref = __ballot_sync(0xffffffffu, (sv & LB_FLAG_MASK) == LB_FLAG_PREFIX);
      if (lane == 0) s_first[warp] = pref ? warp * 32u + (uint32_t)(__ffs(pref) - 1) : 0xFFFFFFFFu;
      __syncthreads();
      uint32_t first = 0xFFFFFFFFu;
#pragma unroll
      for (int w = 0; w < SEL_THREADS / 32; ++w) first = min(first, s_first[w]);
      uint64_t v = tid <= first ? (sv & LB_VALUE_MASK) : 0ull;
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
      if (lane == 0) s_sum[warp] = v;
      __syncthreads();
#pragma unroll
      for (int w = 0; w < SEL_THREADS / 32; ++w) excl += s_sum[w];
      __syncthreads();
      if (first != 0xFFFFFFFFu) break;
      p -= SEL_THREADS;
    }
    if (tid == 0) st_relaxed_u64(status + tile, LB_FLAG_PREFIX | (excl + block_sum));
  }
  if (wcount) {
    uint32_t o = out0 + (uint32_t)excl + warp_excl;
    const uint32_t lt = lanemask_lt();
#pragma unroll
    for (int j = 0; j < SEL_ITEMS; ++j) {
      if ((bal[j] >> lane) & 1u) {
        const uint32_t i = wbase + j * 32;
        const uint64_t key = __ldcg(keys + i);
        const uint32_t at = o + __popc(bal[j] & lt);
        keys_out[at] = key;
        vals_out[at] = i;
        if (list_out) list_out[at] = i;
        const uint32_t w = (uint32_t)key;
#pragma unroll
        for (int d = 0; d < DS_PASSES; ++d) atomicAdd(&s_hist[d * DS_RADIX + ((w >> ds_shift(d)) & ((1u << ds_bits(d)) - 1u))], 1u);
      }
      o += __popc(bal[j]);
    }
  }
  __syncthreads();
  if (block_sum) {
#pragma unroll
    for (int k = 0; k < DS_PASSES * DS_RADIX / SEL_THREADS; ++k) {
      const uint32_t v = s_hist[k * SEL_THREADS + tid];
      if (v) atomicAdd(&region[k * SEL_THREADS + tid], v);
    }
  }
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    s_last = atomicAdd(region + DH_COUNTER, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  // the last CTA: exclusive digit prefixes (thread t owns bin t) and the control block of the class's passes
  uint32_t total = 0;
  for (int d = 0; d < DS_PASSES; ++d) {
    const uint32_t v = tid < (1u << ds_bits(d)) ? __ldcg(region + d * DS_RADIX + tid) : 0u;
    uint32_t in2 = v;
#pragma unroll
    for (int q = 1; q < 32; q <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, in2, q);
      if (lane >= q) in2 += t;
    }
    if (lane == 31) s_warp[warp] = in2;
    __syncthreads();
    uint32_t wex = 0, all = 0;
    for (uint32_t w = 0; w < SEL_THREADS / 32; ++w) {
      if (w < warp) wex += s_warp[w];
      all += s_warp[w];
    }
    if (tid < (1u << ds_bits(d))) region[d * DS_RADIX + tid] = wex + in2 - v;
    total = all;
    __syncthreads();
  }
  if (tid == 0) {
    DepthCtl* ctl = reinterpret_cast<DepthCtl*>(region + DH_CTL);
    ctl->survivors = total;
    uint32_t side = out_side;
    for (int d = 0; d < DS_PASSES; ++d) {
      // the three 9-bit passes always run (the host fixes the final buffer before it knows the digits); the top digit's
      // only if preprocess saw a key of 2^27 or beyond in the class
      const uint32_t skip = d < 3 ? 0u : ((BACK ? fc->top_back : fc->top_front) ? 0u : 1u);
      ctl->skip[d] = skip;
      ctl->in_side[d] = side;
      side ^= skip ^ 1u;
    }
    ctl->final_side = side;
  }
}

// LOOP: the launch is smaller than the number of tiles (which only the device knows: ctl->survivors); its CTAs take
// tickets until the pairs run out. only_if (LOOP): nothing to do when *only_if == 0.
template <int THREADS, int ITEMS, int BITS, bool FIRST, bool LOOP>
__device__ __forceinline__ void
depth_pass_body(uint64_t* __restrict__ keys_a, uint32_t* __restrict__ vals_a, uint64_t* __restrict__ keys_b,
                uint32_t* __restrict__ vals_b, uint32_t n, int pass, int shift, const DepthCtl* __restrict__ ctl,
                const uint32_t* __restrict__ hist_excl, uint64_t* __restrict__ lookback, uint32_t* __restrict__ ticket);

template <int THREADS, int ITEMS, int BITS, int MINB, bool FIRST, bool LOOP>
__global__ void __launch_bounds__(THREADS, MINB)
depth_pass_kernel(uint64_t* __restrict__ keys_a, uint32_t* __restrict__ vals_a, uint64_t* __restrict__ keys_b,
                  uint32_t* __restrict__ vals_b, uint32_t n /* pairs in buffer a (FIRST) */, int pass, int shift,
                  const DepthCtl* __restrict__ ctl, const uint32_t* __restrict__ hist_excl /* [512] this pass */,
                  uint64_t* __restrict__ lookback /* [tiles][1 << BITS], zeroed */, uint32_t* __restrict__ ticket /* zeroed */,
                  const uint32_t* __restrict__ only_if) {
  pdl_launch_dependents();
  pdl_wait();
  if (LOOP && only_if && *only_if == 0u) return;
  depth_pass_body<THREADS, ITEMS, BITS, FIRST, LOOP>(keys_a, vals_a, keys_b, vals_b, n, pass, shift, ctl, hist_excl, lookback, ticket);
}

template <int THREADS, int ITEMS, int BITS, bool FIRST, bool LOOP>
__device__ __forceinline__ void
depth_pass_body(uint64_t* __restrict__ keys_a, uint32_t* __restrict__ vals_a, uint64_t* __restrict__ keys_b,
                uint32_t* __restrict__ vals_b, uint32_t n, int pass, int shift, const DepthCtl* __restrict__ ctl,
                const uint32_t* __restrict__ hist_excl, uint64_t* __restrict__ lookback, uint32_t* __restrict__ ticket) {
  using Core = RadixCore<THREADS, ITEMS, BITS>;
  constexpr int TILE = Core::TILE;
  constexpr uint32_t MASK = (1u << BITS) - 1u;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  OnesweepSmem<THREADS, ITEMS, BITS>& s = *reinterpret_cast<OnesweepSmem<THREADS, ITEMS, BITS>*>(smem_raw);
  if (!FIRST) {
    if (ctl->skip[pass]) return;
    n = ctl->survivors;
  }
  const bool from_a = FIRST || ctl->in_side[pass] == 0u;
  const uint64_t* keys_in = from_a ? keys_a : keys_b;
  const uint32_t* vals_in = from_a ? vals_a : vals_b;
  uint64_t* keys_out = from_a ? keys_b : keys_a;
  uint32_t* vals_out = from_a ? vals_b : vals_a;

  do {
  const uint32_t tile = Core::take_ticket(s.core, ticket);
  const uint32_t tile_base = tile * TILE;
  if (tile_base >= n) return;   // launched for n pairs, S are left: nobody looks back at a tile past the end
  const uint32_t tile_n = min((uint32_t)TILE, n - tile_base);
  const uint32_t tid = threadIdx.x;
  const uint32_t wbase = (tid >> 5) * (ITEMS * 32) + (tid & 31u);
  const uint64_t* kp = keys_in + tile_base + wbase;
  const uint32_t* vp = vals_in + tile_base + wbase;
  uint64_t key[ITEMS];
  uint32_t val[ITEMS], dp[ITEMS];
#pragma unroll
  for (int j = 0; j < ITEMS; ++j) {
    const bool ok = wbase + j * 32 < tile_n;
    key[j] = ok ? __ldcg(kp + j * 32) : ~0ull;
    // FIRST: the pairs come from preprocess in index order, the value of pair i is i
    val[j] = FIRST ? tile_base + wbase + j * 32 : (ok ? __ldcg(vp + j * 32) : 0u);
  }
#pragma unroll
  for (int j = 0; j < ITEMS; ++j) {
    const uint32_t w = (uint32_t)key[j];
    // the culled Gaussians (and the padding of the last tile) carry 0xFFFFFFFF: no element
    dp[j] = w == 0xFFFFFFFFu ? Core::INVALID : ((w >> shift) & MASK);
  }
  // (a wider look-back window for the small front sort was measured and lost: 16 words 0.057 ms for the three passes,
  // 8 words 0.050, 4 words 0.042 -- the words of a 9-bit digit row are 4 KB apart, a window is that many L2 requests)
  Core::template rank<true>(s.core, tile, dp, hist_excl, lookback);
#pragma unroll
  for (int j = 0; j < ITEMS; ++j)
    if (dp[j] != Core::INVALID) {
      s.keys[dp[j] >> Core::DSHIFT] = key[j];
      s.vals[dp[j] >> Core::DSHIFT] = val[j];
    }
  __syncthreads();
  const uint32_t total = s.core.total;
  for (uint32_t p = tid; p < total; p += THREADS) {
    const uint64_t k = s.keys[p];
    const uint32_t o = s.core.out_base[((uint32_t)k >> shift) & MASK] + p;
    keys_out[o] = k;
    vals_out[o] = s.vals[p];
  }
  if (LOOP) __syncthreads();   // the next tile reuses the shared memory
  } while (LOOP);
}

// ---- digit pass over the compact instance payload -----------------------------------------
// When the Gaussians were depth-sorted before duplication, the low 32 key bits of the
// instances are already in order and are dead payload for the remaining tile-id passes, so
// an instance travels as (u16 tile id, u32 Gaussian index): 6 B instead of 12 B. The LAST
// pass writes the indices only -- the tile of a position in the sorted list is implied by
// the tile ranges. (tile << 32 | depth bits) is rebuilt on demand for the debug view.
template <int THREADS, int ITEMS, int BITS>
struct CompactSmem {
  typename RadixCore<THREADS, ITEMS, BITS>::Smem core;
  uint32_t vals[THREADS * ITEMS];
  uint16_t tiles[THREADS * ITEMS];
};

template <int THREADS, int ITEMS, int BITS, int MINB, bool LAST>
__global__ void __launch_bounds__(THREADS, MINB)
compact_pass_kernel(const uint16_t* __restrict__ tiles_in, const uint32_t* __restrict__ vals_in,
                    uint16_t* __restrict__ tiles_out, uint32_t* __restrict__ vals_out, uint32_t n, int shift,
                    const uint32_t* __restrict__ hist_excl, uint64_t* __restrict__ lookback,
                    uint32_t* __restrict__ ticket) {
  using Core = RadixCore<THREADS, ITEMS, BITS>;
  constexpr int TILE = Core::TILE;
  constexpr uint32_t MASK = (1u << BITS) - 1u;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  CompactSmem<THREADS, ITEMS, BITS>& s = *reinterpret_cast<CompactSmem<THREADS, ITEMS, BITS>*>(smem_raw);

  const uint32_t tile = Core::take_ticket(s.core, ticket);
  const uint32_t tile_base = tile * TILE;
  const uint32_t tile_n = min((uint32_t)TILE, n - tile_base);
  const uint32_t tid = threadIdx.x;
  const uint32_t wbase = (tid >> 5) * (ITEMS * 32) + (tid & 31u);
  const uint16_t* tp = tiles_in + tile_base + wbase;
  const uint32_t* vp = vals_in + tile_base + wbase;
  uint32_t t[ITEMS], val[ITEMS], dp[ITEMS];
  if (tile_n == TILE) {
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) t[j] = __ldcs(tp + j * 32);
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) val[j] = __ldcs(vp + j * 32);
  } else {
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const bool ok = wbase + j * 32 < tile_n;
      t[j] = ok ? (uint32_t)__ldcs(tp + j * 32) : 0xFFFFu;   // padding ranks last
      val[j] = ok ? __ldcs(vp + j * 32) : 0u;
    }
  }
#pragma unroll
  for (int j = 0; j < ITEMS; ++j) dp[j] = (t[j] >> shift) & MASK;
  Core::rank(s.core, tile, dp, hist_excl, lookback);
#pragma unroll
  for (int j = 0; j < ITEMS; ++j) {
    s.tiles[dp[j] >> 8] = (uint16_t)t[j];
    s.vals[dp[j] >> 8] = val[j];
  }
  __syncthreads();
  for (uint32_t p = tid; p < tile_n; p += THREADS) {
    const uint32_t tl = s.tiles[p];
    const uint32_t o = s.core.out_base[(tl >> shift) & MASK] + p;
    if (!LAST) tiles_out[o] = (uint16_t)tl;
    vals_out[o] = s.vals[p];
  }
}

// debug view: (tile << 32 | depth bits) of the compact payload
__global__ void __launch_bounds__(256)
keys_from_tiles16_kernel(const uint16_t* __restrict__ tiles16, const uint32_t* __restrict__ vals,
                         const uint4* __restrict__ tileinfo, uint32_t M, uint64_t* __restrict__ keys) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < M) keys[i] = ((uint64_t)tiles16[i] << 32) | tileinfo[vals[i]].z;
}

__global__ void __launch_bounds__(256)
keys_from_ranges_kernel(const uint2* __restrict__ ranges, const uint32_t* __restrict__ vals,
                        const uint4* __restrict__ tileinfo, uint64_t* __restrict__ keys) {
  const uint2 r = ranges[blockIdx.x];
  for (uint32_t i = r.x + threadIdx.x; i < r.y; i += blockDim.x)
    keys[i] = ((uint64_t)blockIdx.x << 32) | tileinfo[vals[i]].z;
}

}  // namespace pvg

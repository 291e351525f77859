// blend.cuh -- stage a5: per-tile front-to-back alpha compositing
//   C = sum_i T_i alpha_i c_i,  T_i = prod_{j<i} (1 - alpha_j)      (Eq. 3)
//   alpha = min(0.99, o~ * exp(-1/2 d^T Sigma'^-1 d))
//   depth = sum T alpha z / sum T alpha, O = sum T alpha
// with the 1/255 alpha cutoff, the 0.99 clamp and the T < 1e-4 stop (S9, S10).
// FP32-pipe bound: no tensor cores (not a dense contraction).
#pragma once

#include "common.cuh"

namespace pvg {

#ifndef PVG_BLEND_NPX
#define PVG_BLEND_NPX 4
#endif
constexpr int BLEND_NPX = PVG_BLEND_NPX;                   // horizontally adjacent pixels per thread (2 or 4)
constexpr int BLEND_THREADS = PVG_TILE_PIXELS / BLEND_NPX;
#ifndef PVG_BLEND_BATCH
#define PVG_BLEND_BATCH 128
#endif
constexpr int BLEND_BATCH = PVG_BLEND_BATCH;   // 88 B of (duplicated) shared memory per staged entry
#ifndef PVG_BLEND_FIRST
#define PVG_BLEND_FIRST 128
#endif
constexpr int BLEND_BATCH_FIRST = PVG_BLEND_FIRST;
#ifndef PVG_BLEND_UNROLL
#define PVG_BLEND_UNROLL 4
#endif
constexpr int BLEND_UNROLL = PVG_BLEND_UNROLL;   // divides BLEND_BATCH_FIRST / (BLEND_THREADS / 32)
#ifndef PVG_BLEND_MINB
#define PVG_BLEND_MINB 12   // resident CTAs per SM the register allocation must allow
#endif

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// f_sky(d) (layout and filter: DESIGN.md S20-S22): face = 2 a + (d_a < 0) with a the axis of
// largest |d_a| (ties: lowest axis), u = d_b / |d_a|, v = d_c / |d_a| for (b, c) the next two axes in cyclic
// order, texel centres at (2 i + 1) / res - 1, bilinear between the four nearest centres, clamped to the face.
__device__ __forceinline__ void sky_sample(const float* __restrict__ cube, int res, float dx, float dy, float dz, float (&out)[3]) {
  const float ax = fabsf(dx), ay = fabsf(dy), az = fabsf(dz);
  int a = 0;
  float m = ax, da = dx, u = dy, v = dz;
  if (ay > m) { a = 1; m = ay; da = dy; u = dz; v = dx; }
  if (az > m) { a = 2; m = az; da = dz; u = dx; v = dy; }
  const int face = 2 * a + (da < 0.f ? 1 : 0);
  const float inv = 1.0f / m;
  const float r = (float)res;
  float sx = fmaf(fmaf(u, inv, 1.0f), 0.5f * r, -0.5f), sy = fmaf(fmaf(v, inv, 1.0f), 0.5f * r, -0.5f);
  sx = fminf(fmaxf(sx, 0.f), r - 1.0f);
  sy = fminf(fmaxf(sy, 0.f), r - 1.0f);
  const int i0 = (int)sx, j0 = (int)sy;   // sx, sy >= 0: truncation is the floor
  const int i1 = min(i0 + 1, res - 1), j1 = min(j0 + 1, res - 1);
  const float fx = sx - (float)i0, fy = sy - (float)j0;
  const float* F = cube + (size_t)face * res * res * 3;
  const float* p00 = F + ((size_t)j0 * res + i0) * 3;
  const float* p10 = F + ((size_t)j0 * res + i1) * 3;
  const float* p01 = F + ((size_t)j1 * res + i0) * 3;
  const float* p11 = F + ((size_t)j1 * res + i1) * 3;
#pragma unroll
  for (int ch = 0; ch < 3; ++ch) {
    const float top = fmaf(fx, __ldg(p10 + ch) - __ldg(p00 + ch), __ldg(p00 + ch));
    const float bot = fmaf(fx, __ldg(p11 + ch) - __ldg(p01 + ch), __ldg(p01 + ch));
    out[ch] = fmaf(fy, bot - top, top);
  }
}

// Can the Gaussian reach alpha >= 1/255 at any pixel centre of the box [x0, x1] x [y0, y1]? Its exponent
// w(x) = a' dx^2 + b' dx dy + c' dy^2 + L (log2 units; a', c' < 0, concave) is maximised over the box: 0 + L if
// the centre is inside, else on one of the four edges at the clamped stationary point of the 1-D restriction.
// Conservative: the margin covers the fp32 rounding of this evaluation and of the per-pixel one (a few ulps
// of the sum of the term magnitudes, which cancel for needles) and ex2.approx; anything non-finite keeps.
__device__ __forceinline__ bool blend_reaches_tile(float mx, float my, float a, float b, float c, float L,
                                                   float x0, float x1, float y0, float y1) {
  const float dx0 = x0 - mx, dx1 = x1 - mx, dy0 = y0 - my, dy1 = y1 - my;
  if (dx0 <= 0.f && dx1 >= 0.f && dy0 <= 0.f && dy1 >= 0.f) return true;
  const float hb_c = -0.5f * b / c, hb_a = -0.5f * b / a;   // stationary dy per dx, dx per dy
  float best = -3.0e38f;
#pragma unroll
  for (int e = 0; e < 2; ++e) {
    const float dx = e ? dx1 : dx0;
    const float dy = fminf(fmaxf(hb_c * dx, dy0), dy1);
    best = fmaxf(best, fmaf(fmaf(a, dx, b * dy), dx, (c * dy) * dy));
    const float ey = e ? dy1 : dy0;
    const float ex = fminf(fmaxf(hb_a * ey, dx0), dx1);
    best = fmaxf(best, fmaf(fmaf(a, ex, b * ey), ex, (c * ey) * ey));
  }
  const float Dx = fmaxf(fabsf(dx0), fabsf(dx1)), Dy = fmaxf(fabsf(dy0), fabsf(dy1));
  const float S = fabsf(a) * Dx * Dx + fabsf(b) * Dx * Dy + fabsf(c) * Dy * Dy;
  const float bound = L + best + fmaf(S, 2e-6f, 1e-3f);
  return !(bound < -7.994353436858858f);   // log2(1/255); NaN keeps
}

// ---- packed fp32 (sm_100: add / sub / mul / fma .f32x2 on 64-bit register pairs) -------------------------------
// The kernel is ISSUE-bound (ncu, round 1: issue-active 84 %, 18 instructions per (pixel, entry) evaluation; round 2
// confirmed it: trading ALU-pipe instructions for FMA-pipe ones one for one left the time unchanged). A packed
// instruction performs the fp32 operation on both halves of a register pair -- the SAME IEEE operation per half,
// so results are bit-identical to the scalar form -- for ONE issue slot. pvg_calibrate_fp32 measures what it buys:
// FFMA2 issues at half the FFMA rate, i.e. the same FMAs per second, but leaves every other slot to the compares,
// selects, MUFU and shared-memory loads that make up the rest of this loop. A thread's four pixels form two pairs.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
  f32x2 v;
  asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(lo), "f"(hi));
  return v;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
  f32x2 d;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) {
  f32x2 d;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}

// Compositing state of a PAIR of horizontally adjacent pixels and one front-to-back step.
//   * no `alive` predicate: a stopped pixel carries its final transmittance NEGATED (T < 0). Then T' = T - alpha T
//     < 0 fails `T' >= 1e-4` by itself, nothing is ever composited again, and the stop is idempotent;
//   * the contribution is added unconditionally with a weight that is 0 unless the entry is composited
//     (fma(c, 0, C) = C exactly: colours and depths are finite), so that the five accumulations are packed;
//   * the two clamps -- w <= log2 o~ (S16': the exact quadratic form is <= 0) and alpha <= 0.99 -- are applied only to
//     entries that can need them (decided per entry by the staging code, below).
struct BlendPair {
  f32x2 T, Cr, Cg, Cb, D;   // T > 0: live; T < 0: stopped, |T| final (outside the image: -1)
  // alpha of the entry at the two pixels (clamps applied); r2 .. z2: the entry's colour and depth, each duplicated
  template <bool WANT_FLAG>
  __device__ __forceinline__ uint32_t step(float a0, float a1, f32x2 r2, f32x2 g2, f32x2 b2, f32x2 z2) {
    // T' = T (1 - alpha) with 1 - alpha formed off the T -> T' recurrence: the loop-carried chain of a pixel is
    // FMUL2 -> FSETP -> FSEL (the profile of the T - alpha T form showed its FMUL2 -> FADD2 pair as the top stall)
    const f32x2 al = pack2(a0, a1);
    const f32x2 wg = mul2(al, T);                                     // alpha T: the weight of the contribution
    const f32x2 tn = mul2(T, sub2(0x3f8000003f800000ull, al));        // (1.0f, 1.0f) - alpha
    float t0, t1, g0, g1, n0, n1;
    unpack2(T, t0, t1);
    unpack2(wg, g0, g1);
    unpack2(tn, n0, n1);
    const bool pa0 = a0 >= PVG_ALPHA_MIN, pa1 = a1 >= PVG_ALPHA_MIN;      // listed (false for NaN)
    const bool pu0 = pa0 && n0 >= PVG_T_STOP, pu1 = pa1 && n1 >= PVG_T_STOP;   // composited; listed and not composited: stop (S10)
    const f32x2 we = pack2(pu0 ? g0 : 0.f, pu1 ? g1 : 0.f);
    Cr = fma2(r2, we, Cr);
    Cg = fma2(g2, we, Cg);
    Cb = fma2(b2, we, Cb);
    D = fma2(z2, we, D);
    T = pack2(pa0 ? (pu0 ? n0 : -fabsf(t0)) : t0, pa1 ? (pu1 ? n1 : -fabsf(t1)) : t1);
    return WANT_FLAG ? (pu0 ? 1u : 0u) + (pu1 ? 1u : 0u) : 0u;
  }
};

// One CTA per 16x16 tile, one thread per BLEND_NPX horizontally adjacent pixels (they share dy and
// with it 4 of the operations of the exponent, and every shared-memory load). The tile's slice
// of the sorted instance list is consumed in batches: each thread gathers 48 B records through the
// sorted index list into shared memory, pre-digested so that the inner loop is straight-line:
//   conic scaled by -log2(e)/2 and log2(o~) carried as the constant term, so that
//   alpha = min(0.99, ex2(a' dx^2 + b' dx dy + c' dy^2 + log2 o~)) needs no multiply by o~.
// The per-pixel decisions (1/255 cutoff, T stop) are predicates, not branches: 71% of the
// evaluations contribute at config 3, so a warp practically always has a contributing lane and
// branching only added reconvergence overhead. A warp leaves the batch as soon as none of its
// pixels is alive; the tile retires when every pixel's transmittance has dropped below 1e-4.
// COUNT = true additionally counts the (pixel, list entry) evaluations reached and the
// contributing ones into counters[0..1] (measurement only, never on the product path).
// MODE: BLEND_COLOR -- rgb = C + T bg, depth = D / (1 - T); BLEND_SKY -- the background is the cube map f_sky(d)
// (its own instantiation, so that the lookup's registers do not cost the plain kernel occupancy);
// BLEND_FEATURE -- "flexible rendering": the record's colour slot holds another per-Gaussian
// quantity (here vbar in camera axes) and `featw` a fourth one (clamp(rho, 0, 2)); the outputs are the plain sums
// sum T alpha f of Eq. 3, without background and without normalisation, in out_rgb and out_depth.
enum { BLEND_COLOR = 0, BLEND_SKY = 1, BLEND_FEATURE = 2 };

// Lazy lists (blockbin.cuh, PVG_OPT_LAZY_CHUNKS): a tile's list is first written only as far as the first c0
// chunks of its block reach; most tiles saturate inside that prefix and the rest of their list is never needed.
//   PHASE 0: the whole list at once (the lists are complete).
//   PHASE 1: the prefix [begin, lim). A tile that still has a live pixel at lim < end parks its per-pixel state
//            (T, C, D; the sign of T carries `alive`) and marks itself in unf_tile / unf_mask; every other tile
//            writes its pixels.
//   PHASE 2: only the marked tiles: they take their state back and go on from lim to the end, by then written
//            by the second bin_write round. Same entries, same order, same arithmetic: the image is bit-identical.
// lim[tile] is the position after chunk min(c0, chunks of the block) - 1 of the tile's block, stored by the warp
// of bin_write's first round that owns that chunk. Phase 2 is a persistent launch over the list of parked tiles.
struct BlendLazy {
  const uint32_t* lim;             // [tiles] end of the written prefix of every non-empty list (bin_write, round 0)
  float* state;                    // [5][H * W]
  unsigned long long* unf_mask;    // [blocks] bit (ty & 7) * 8 + (tx & 7), zeroed
  uint32_t* unf_count;             // [1] zeroed: number of parked tiles
  uint32_t* unf_list;              // [tiles] the parked tiles, in parking order
  volatile uint64_t* parked_host;  // mapped host word: the count, for pvg_frame_stats
  uint32_t blocks_x;
};

// The second round of the lazy lists, launched FROM THE DEVICE (round2.cuh, round2.cu): the launch parameters of its
// kernels, filled by the host before the first blend phase. After that phase a one-thread gate kernel reads the
// parked count; if it is not zero it tail-launches the chain (CUDA dynamic parallelism: the kernels run in order once
// the gate has completed, and whatever the host enqueued next runs after them). A frame in which no tile parked --
// the normal case -- then pays one small launch for the second round, where nine launches that found nothing to do
// cost 25-35 us.
struct FrontCtl;   // onesweep.cuh
struct R2Chain {
  uint32_t enabled;      // 0: the host launches the second round itself (PVG_R2_TAIL=0)
  // the back of the depth order (front-first, onesweep.cuh): select, passes, scan
  uint32_t back;
  const uint64_t* okeys; uint32_t n; const FrontCtl* fc;
  uint64_t* sel_keys; uint32_t* sel_vals; uint32_t* sel_region; uint64_t* sel_status; uint32_t* sel_ticket;
  uint32_t sel_side, sel_grid;
  uint64_t* lb; uint32_t lb_rows, lb_tile;
  uint64_t *ka, *kb; uint32_t *va, *vb;
  uint32_t back_count, passes, pass_grid; uint32_t* pass_tickets;
  uint32_t scan_grid; const uint64_t* scan_keys; const uint32_t* visit; uint32_t* boffsets; uint64_t* scan_total;
  uint64_t* scan_status; uint32_t* scan_ticket; uint32_t* chunk_owner; uint32_t owner_chunk, rank0; const uint64_t* scan_init;
  const uint32_t* counts;
  // the records of the whole scene
  uint32_t shade, shade_grid; const float4 *A0, *A1, *A2, *A3, *SH; float4* record; float* featw;
  // the entries behind the first slab
  uint32_t emit, emit_grid, emit_bits, nv, Mb, blocks_x, emit_tiles;
  uint32_t* s_g; uint64_t* s_mask; const uint32_t* bin_start; uint64_t* emit_lookback; uint32_t* emit_ticket;
  // the rest of the parked tiles' lists
  uint32_t write_grid; const uint2* ranges; uint32_t tiles_x, tiles_y; uint64_t* chunk_cnt; uint32_t* write_ticket;
  uint32_t* vals; uint32_t kin_lo; const unsigned long long* want_mask; const uint32_t* want_count; const uint64_t* avail;
  // the second blend phase
  uint32_t blend_grid;
};
// Parks a tile (first blend phase of the lazy lists): out of line, so that the rare path costs the common one nothing.
// st[k] = (T signed: negative = stopped, Cr, Cg, Cb, D).
__device__ __noinline__ void blend_park(const BlendLazy& Z, uint32_t tile, uint32_t bin, uint32_t ltile, size_t HW, size_t pi,
                                        uint32_t inmask, const float (&st)[BLEND_NPX][5]) {
#pragma unroll
  for (int k = 0; k < BLEND_NPX; ++k) {
    if (!((inmask >> k) & 1u)) continue;
#pragma unroll
    for (int c = 0; c < 5; ++c) Z.state[c * HW + pi + k] = st[k][c];
  }
  if (threadIdx.x == 0) {
    Z.unf_list[atomicAdd(Z.unf_count, 1u)] = tile;
    atomicOr(Z.unf_mask + bin, 1ull << ltile);
  }
}

// log2(0.98): entries with o~ above it take the clamped evaluation (the 0.99 clamp can bind only above log2 0.99;
// the margin covers the rounding of w)
#define PVG_L_CLAMPED -0.029146346f

template <bool COUNT, int MODE, int PHASE>
__device__ __forceinline__ void
blend_tile(const FrameParams& P, const uint32_t tile, const uint2* __restrict__ ranges,
           const uint32_t* __restrict__ vals, const float4* __restrict__ record,
           float* __restrict__ out_rgb, float* __restrict__ out_depth, float* __restrict__ out_alpha,
           unsigned long long* __restrict__ counters, const float* __restrict__ featw, const BlendLazy& Z) {
  // every per-entry operand of a packed instruction is stored DUPLICATED, so that one 128-bit shared-memory load
  // fills two register pairs and no instruction is spent on broadcasting
  __shared__ float4 s_xa[BLEND_BATCH];    // mx, mx, a', a'
  __shared__ float4 s_yb[BLEND_BATCH];    // my, my, b', b'
  __shared__ float4 s_cl[BLEND_BATCH];    // c', c', log2 o~, log2 o~
  __shared__ float4 s_rg[BLEND_BATCH];    // r, r, g, g
  __shared__ float4 s_bz[BLEND_BATCH];    // b, b, z, z
  __shared__ float2 s_clamp[BLEND_BATCH]; // upper clamp of w (+inf: none), upper clamp of alpha (+inf: none)
  __shared__ uint32_t s_kept[BLEND_THREADS / 32];
  __shared__ uint32_t s_plain[BLEND_BATCH / BLEND_UNROLL];   // per group of BLEND_UNROLL staged entries: none of them is clamped

  const uint32_t tid = threadIdx.x;
  const uint32_t tx = tile % P.tiles_x, ty = tile / P.tiles_x;
  constexpr uint32_t TPR = PVG_TILE / BLEND_NPX;   // threads per tile row
  const uint32_t px = tx * PVG_TILE + BLEND_NPX * (tid % TPR), py = ty * PVG_TILE + tid / TPR;
  const float pxf = (float)px + 0.5f, pyf = (float)py + 0.5f;   // S14
  uint2 range = ranges[tile];
  const uint32_t list_end = range.y;
  (void)list_end;
  if (PHASE != 0) {
    // lim[] is zeroed: a tile whose block has no complete chunk yet stands at its list's begin
    const uint32_t lim = range.x == range.y ? range.y : max(Z.lim[tile], range.x);
    if (PHASE == 1) range.y = lim; else range.x = lim;
  }

  static_assert(BLEND_NPX == 4 || BLEND_NPX == 8, "two or four pixel pairs per thread");
  constexpr int NPAIR = BLEND_NPX / 2;
  BlendPair X[NPAIR];
  {
    float st[BLEND_NPX][5];
#pragma unroll
    for (int k = 0; k < BLEND_NPX; ++k) {
      const bool in = px + k < (uint32_t)P.width && py < (uint32_t)P.height;
      st[k][0] = in ? 1.f : -1.f;
      st[k][1] = st[k][2] = st[k][3] = st[k][4] = 0.f;
      if (PHASE == 2 && in) {
        const size_t HW = (size_t)P.width * P.height;
        const size_t pi = (size_t)py * P.width + px;
#pragma unroll
        for (int c = 0; c < 5; ++c) st[k][c] = Z.state[c * HW + pi + k];
      }
    }
#pragma unroll
    for (int p = 0; p < NPAIR; ++p) {
      X[p].T = pack2(st[2 * p][0], st[2 * p + 1][0]);
      X[p].Cr = pack2(st[2 * p][1], st[2 * p + 1][1]);
      X[p].Cg = pack2(st[2 * p][2], st[2 * p + 1][2]);
      X[p].Cb = pack2(st[2 * p][3], st[2 * p + 1][3]);
      X[p].D = pack2(st[2 * p][4], st[2 * p + 1][4]);
    }
  }
  // a pixel is live while its T is positive: some pixel of the thread is live iff the AND of the four sign bits is clear
  auto any_alive = [&]() {
    f32x2 m = X[0].T;
#pragma unroll
    for (int p = 1; p < NPAIR; ++p) m &= X[p].T;
    return (m & 0x8000000080000000ull) != 0x8000000080000000ull;
  };
  // the pixel centres of the two pairs, and the row, as packed operands
  f32x2 pxp[NPAIR];
#pragma unroll
  for (int p = 0; p < NPAIR; ++p) pxp[p] = pack2(pxf + (float)(2 * p), pxf + (float)(2 * p + 1));
  const f32x2 pyp = pack2(pyf, pyf);
  uint32_t n_eval = 0, n_contrib = 0;

  // The tile's box of pixel centres, for the staging-time test below.
  const float bx0 = (float)(tx * PVG_TILE) + 0.5f, bx1 = bx0 + (float)(PVG_TILE - 1);
  const float by0 = (float)(ty * PVG_TILE) + 0.5f, by1 = by0 + (float)(PVG_TILE - 1);
  const uint32_t lane = tid & 31u, wid = tid >> 5;
  constexpr uint32_t WARPS = BLEND_THREADS / 32;
  const float kInf = __int_as_float(0x7f800000);

  // One group of BLEND_UNROLL staged entries (slots j .. j + 3, of which the first `real` are list entries and the
  // rest padding) against the thread's two pixel pairs. PLAIN: no entry of the group is clamped; otherwise the plain
  // evaluation plus two FMNMX per pixel, which are no-ops on the group's unclamped entries (their clamps are +inf).
  auto group = [&]<bool PLAIN>(uint32_t j, uint32_t real) {
#pragma unroll
    for (int u = 0; u < BLEND_UNROLL; ++u) {
      const ulonglong2 xa = *reinterpret_cast<const ulonglong2*>(&s_xa[j + u]);
      const ulonglong2 yb = *reinterpret_cast<const ulonglong2*>(&s_yb[j + u]);
      const ulonglong2 cl = *reinterpret_cast<const ulonglong2*>(&s_cl[j + u]);
      const ulonglong2 rg = *reinterpret_cast<const ulonglong2*>(&s_rg[j + u]);
      const ulonglong2 bz = *reinterpret_cast<const ulonglong2*>(&s_bz[j + u]);
      // log2 of o~ exp(-1/2 (a dx^2 + c dy^2) - b dx dy) = dx (a' dx + b' dy) + (c' dy^2 + log2 o~); both halves
      // of every row term hold the same value
      const f32x2 dy = sub2(yb.x, pyp);
      const f32x2 q = mul2(yb.y, dy);
      const f32x2 rr = fma2(mul2(cl.x, dy), dy, cl.y);
      float2 clamp = make_float2(0.f, 0.f);
      if (!PLAIN) clamp = s_clamp[j + u];
#pragma unroll
      for (int p = 0; p < NPAIR; ++p) {
        if (COUNT) {
          float t0, t1;
          unpack2(X[p].T, t0, t1);
          n_eval += ((uint32_t)u < real ? 1u : 0u) * ((t0 > 0.f ? 1u : 0u) + (t1 > 0.f ? 1u : 0u));
        }
        const f32x2 dx = sub2(xa.x, pxp[p]);
        float w0, w1;
        unpack2(fma2(fma2(xa.y, dx, q), dx, rr), w0, w1);
        if (!PLAIN) { w0 = fminf(w0, clamp.x); w1 = fminf(w1, clamp.x); }   // S16'
        float a0 = ex2_approx(w0), a1 = ex2_approx(w1);
        if (!PLAIN) { a0 = fminf(a0, clamp.y); a1 = fminf(a1, clamp.y); }   // S9
        const uint32_t used = X[p].template step<COUNT>(a0, a1, rg.x, rg.y, bz.x, bz.y);
        if (COUNT) n_contrib += used;
      }
    }
  };

  // batches grow 64 -> 128 -> 256: at config 3 a tile consumes ~90 entries on average before it
  // saturates, so a fixed 256-entry first batch gathers mostly records that are never used
  uint32_t bs = BLEND_BATCH_FIRST;
  uint32_t base = range.x;   // after the loop: base < range.y iff it ended because every pixel of the tile had stopped
  for (; base < range.y; base += bs, bs = min(2u * bs, (uint32_t)BLEND_BATCH)) {
    // all pixels of the tile saturated? (also fences the previous batch's smem reads)
    if (__syncthreads_count(any_alive()) == 0) break;
    // Staging. Warp w gathers the w-th segment of the batch and keeps, in order, only the entries whose
    // ellipse { alpha >= 1/255 } can reach the tile at all: the lists are built from axis-aligned
    // rectangles (S7), and 26% (config 3) to 48% (config 4) of the entries a tile consumes cover it with
    // their rectangle only. A dropped entry would have been rejected at every pixel, so the image is
    // unchanged bit for bit (blend_reaches_tile is conservative by a margin).
    const uint32_t seg = bs / WARPS, seg0 = wid * seg;
    uint32_t kept = 0;
    for (uint32_t r = 0; r < seg; r += 32) {
      const uint32_t idx = base + seg0 + r + lane;
      bool keep = false;
      float4 ge, co, bz;   // (mx, my, a', b'), (c', log2 o~, r, g), (b, z, clamp of w, clamp of alpha)
      if (idx < range.y) {
        const uint32_t g = __ldg(vals + idx);
        const float4 r0 = __ldg(record + 3 * (size_t)g);
        const float4 r1 = __ldg(record + 3 * (size_t)g + 1);
        const float4 r2 = __ldg(record + 3 * (size_t)g + 2);
        const float kh = -0.72134752044448170f;  // -log2(e)/2
        ge = make_float4(r0.x, r0.y, kh * r1.x, 2.0f * kh * r1.y);
        co = make_float4(kh * r1.z, __log2f(r0.w), r2.x, r2.y);
        // Which entries need the clamps evaluated (a property of the entry alone, so that a (pixel, entry) evaluation
        // does not depend on how the list was cut into batches): alpha <= 0.99 can only bind when o~ is near 1, and
        // w <= log2 o~ holds up to rounding whenever the conic is positive definite with a margin in fp32
        // (4 a' c' - b'^2 = 4 kh^2 (a c - b^2)); everything else -- needles whose rounded conic is indefinite, NaN --
        // takes the clamped path.
        const bool safe = co.y <= PVG_L_CLAMPED && 4.0f * ge.z * co.x > 1.00001f * ge.w * ge.w;
        bz = make_float4(r2.z, MODE == BLEND_FEATURE ? __ldg(featw + g) : r0.z, safe ? kInf : co.y, safe ? kInf : PVG_ALPHA_MAX);
        keep = !P.cull || blend_reaches_tile(ge.x, ge.y, ge.z, ge.w, co.x, co.y, bx0, bx1, by0, by1);
      }
      const uint32_t m = __ballot_sync(0xffffffffu, keep);
      if (keep) {
        const uint32_t slot = seg0 + kept + __popc(m & ((1u << lane) - 1u));
        s_xa[slot] = make_float4(ge.x, ge.x, ge.z, ge.z);
        s_yb[slot] = make_float4(ge.y, ge.y, ge.w, ge.w);
        s_cl[slot] = make_float4(co.x, co.x, co.y, co.y);
        s_rg[slot] = make_float4(co.z, co.z, co.w, co.w);
        s_bz[slot] = make_float4(bz.x, bz.x, bz.y, bz.y);
        s_clamp[slot] = make_float2(bz.z, bz.w);
      }
      kept += __popc(m);
    }
    // padding up to the unroll factor: log2 o~ = -inf gives alpha = 0 (kept < seg leaves room: seg % 4 == 0)
    if (lane < ((0u - kept) & (BLEND_UNROLL - 1u))) {
      const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
      s_xa[seg0 + kept + lane] = zero;
      s_yb[seg0 + kept + lane] = zero;
      s_cl[seg0 + kept + lane] = make_float4(0.f, 0.f, __int_as_float(0xff800000), __int_as_float(0xff800000));
      s_rg[seg0 + kept + lane] = zero;
      s_bz[seg0 + kept + lane] = zero;
      s_clamp[seg0 + kept + lane] = make_float2(kInf, kInf);
    }
    if (lane == 0) s_kept[wid] = kept;
    __syncwarp();
    // group flags of this warp's segment (a group is what one trip of the unrolled loop below consumes)
    for (uint32_t gq = lane; BLEND_UNROLL * gq < kept; gq += 32) {
      uint32_t m = 0x7f800000u;
#pragma unroll
      for (int u = 0; u < BLEND_UNROLL; ++u) m &= __float_as_uint(s_clamp[seg0 + BLEND_UNROLL * gq + u].x);
      s_plain[seg0 / BLEND_UNROLL + gq] = m == 0x7f800000u ? 1u : 0u;   // +inf's bit pattern survives the AND iff all four are +inf
    }
    __syncthreads();
    if (__any_sync(0xffffffffu, any_alive())) {
      for (uint32_t sg = 0; sg < WARPS; ++sg) {
        const uint32_t nb = s_kept[sg], j00 = sg * seg;
        bool stop = false;
        for (uint32_t j0 = 0; j0 < nb; j0 += BLEND_UNROLL) {
          // warp-uniform (every lane looks at the same entries): the clamped evaluation is the plain one plus two
          // FMNMX per (pixel, entry), and a no-op on the group's unclamped entries (their clamps are +inf)
          // warp-uniform (every lane looks at the same entries): two copies of the group's code, so that the
          // common one carries no clamp instructions at all
          if (s_plain[(j00 + j0) / BLEND_UNROLL]) group.template operator()<true>(j00 + j0, nb - j0);
          else group.template operator()<false>(j00 + j0, nb - j0);
          if (!__any_sync(0xffffffffu, any_alive())) { stop = true; break; }
        }
        if (stop) break;
      }
    }
  }

  if (COUNT) {
    atomicAdd(counters, (unsigned long long)n_eval);
    atomicAdd(counters + 1, (unsigned long long)n_contrib);
  }
  const size_t HW = (size_t)P.width * P.height;
  const size_t pi = (size_t)py * P.width + px;
  if (PHASE == 1 && base >= range.y && range.y < list_end) {
    // the written prefix is used up without the tile being known dead: park it if a pixel is still alive
    // (block-uniform decision; rare -- a saturating tile leaves the loop through the check at its top)
    if (__syncthreads_or(any_alive())) {
      float st[BLEND_NPX][5];
#pragma unroll
      for (int p = 0; p < NPAIR; ++p) {
        unpack2(X[p].T, st[2 * p][0], st[2 * p + 1][0]);
        unpack2(X[p].Cr, st[2 * p][1], st[2 * p + 1][1]);
        unpack2(X[p].Cg, st[2 * p][2], st[2 * p + 1][2]);
        unpack2(X[p].Cb, st[2 * p][3], st[2 * p + 1][3]);
        unpack2(X[p].D, st[2 * p][4], st[2 * p + 1][4]);
      }
      uint32_t inmask = 0;
#pragma unroll
      for (int k = 0; k < BLEND_NPX; ++k) inmask |= (px + k < (uint32_t)P.width && py < (uint32_t)P.height) ? 1u << k : 0u;
      blend_park(Z, tile, (ty >> 3) * Z.blocks_x + (tx >> 3), (ty & 7u) * 8u + (tx & 7u), HW, pi, inmask, st);
      return;
    }
  }
  float fin[BLEND_NPX][5];
#pragma unroll
  for (int p = 0; p < NPAIR; ++p) {
    unpack2(X[p].T, fin[2 * p][0], fin[2 * p + 1][0]);
    unpack2(X[p].Cr, fin[2 * p][1], fin[2 * p + 1][1]);
    unpack2(X[p].Cg, fin[2 * p][2], fin[2 * p + 1][2]);
    unpack2(X[p].Cb, fin[2 * p][3], fin[2 * p + 1][3]);
    unpack2(X[p].D, fin[2 * p][4], fin[2 * p + 1][4]);
  }
#pragma unroll
  for (int k = 0; k < BLEND_NPX; ++k) {
    if (!(px + k < (uint32_t)P.width && py < (uint32_t)P.height)) continue;   // recomputed: not kept live through the loop
    const float Tk = fabsf(fin[k][0]);
    const float Al = 1.0f - Tk;
    if (out_rgb) {
      float bg[3] = {P.bg[0], P.bg[1], P.bg[2]};
      if (MODE == BLEND_FEATURE) bg[0] = bg[1] = bg[2] = 0.f;
      if (MODE == BLEND_SKY) {
        // the pixel-centre ray in world coordinates: R^T ((x - cx) / fx, (y - cy) / fy, 1)
        const float cxr = (pxf + (float)k - P.cx) / P.fx, cyr = (pyf - P.cy) / P.fy;
        sky_sample(P.sky, P.sky_res, fmaf(P.R[0], cxr, fmaf(P.R[3], cyr, P.R[6])),
                   fmaf(P.R[1], cxr, fmaf(P.R[4], cyr, P.R[7])), fmaf(P.R[2], cxr, fmaf(P.R[5], cyr, P.R[8])), bg);
      }
      out_rgb[pi + k] = fmaf(Tk, bg[0], fin[k][1]);
      out_rgb[HW + pi + k] = fmaf(Tk, bg[1], fin[k][2]);
      out_rgb[2 * HW + pi + k] = fmaf(Tk, bg[2], fin[k][3]);
    }
    if (out_depth) out_depth[pi + k] = MODE == BLEND_FEATURE ? fin[k][4] : (Al > 0.f ? fin[k][4] / Al : 0.f);
    if (out_alpha) out_alpha[pi + k] = Al;
  }
}

template <bool COUNT, int MODE, int PHASE>
__global__ void __launch_bounds__(BLEND_THREADS, PVG_BLEND_MINB)
blend_kernel(const __grid_constant__ FrameParams P, const uint2* __restrict__ ranges,
             const uint32_t* __restrict__ vals, const float4* __restrict__ record,
             float* __restrict__ out_rgb, float* __restrict__ out_depth, float* __restrict__ out_alpha,
             unsigned long long* __restrict__ counters, const float* __restrict__ featw,
             const __grid_constant__ BlendLazy Z) {
  pdl_launch_dependents();
  pdl_wait();
  if (PHASE != 2) {
    // one CTA per tile; only the band's tiles are launched
    blend_tile<COUNT, MODE, PHASE>(P, blockIdx.x + (uint32_t)P.band_y0 * (uint32_t)P.tiles_x, ranges, vals, record, out_rgb,
                                   out_depth, out_alpha, counters, featw, Z);
  } else {
    const uint32_t parked = *Z.unf_count;
    if (blockIdx.x == 0 && threadIdx.x == 0) *Z.parked_host = parked;
    for (uint32_t it = blockIdx.x; it < parked; it += gridDim.x) {
      blend_tile<COUNT, MODE, 2>(P, Z.unf_list[it], ranges, vals, record, out_rgb, out_depth, out_alpha, counters, featw, Z);
      __syncthreads();   // the next tile's staging reuses the shared-memory batch
    }
  }
}

}  // namespace pvg

// preprocess.cuh -- stage a1: per-Gaussian state at time t and its projection.
//
// One thread per Gaussian. HBM-bound: 4 coalesced 128-bit loads of the SoA model
// (64 B), 3..12 more for the SH planes of survivors only (<= 192 B), one 48 B record
// + 16 B tile info + 4 B count out. Steps P1..P12 of DESIGN.md:
//   Eq. 6 mu~(t), Eq. 7 (L105) o~(t) -- or the temporal-smoothing state of Eq. 12 (L162) and
//   the staticness filter on rho = beta / l (L118, L192) --, culls, Sigma from (q, s) (L79),
//   Eq. 2 (L68) EWA projection with 0.3 px^2 dilation, conic, exact-cutoff extents,
//   tile rectangle, degree-3 SH colour viewed from mu~(t).
#pragma once

#include "common.cuh"

namespace pvg {

// real SH constants sqrt(k / (m pi)) (closed forms; evaluated once, offline)
#define SH_C0 0.28209479177387814f
#define SH_C1 0.4886025119029199f
#define SH_C2A 1.0925484305920792f
#define SH_C2B 0.31539156525252005f
#define SH_C2C 0.5462742152960396f
#define SH_C3A 0.5900435899266435f
#define SH_C3B 2.890611442640554f
#define SH_C3C 0.4570457994644658f
#define SH_C3D 0.3731763325901154f
#define SH_C3E 1.445305721320277f

// Model layout in HBM (built once by relayout_kernel):
//   A0[i] = (mu.x, mu.y, mu.z, tau)     A1[i] = (v.x, v.y, v.z, beta)
//   A2[i] = unit quaternion (w,x,y,z)   A3[i] = (s.x, s.y, s.z, o)
//   SH[p][i], p = 0..11: floats 4p..4p+3 of the point's [16][3] coefficient block
// Outputs:
//   record[3 i + {0,1,2}] = (mx,my,z,o~), (a,b,c,hx), (r,g,b,hy)   -- all 0 if culled; with P.target == 1 the
//                           colour slot holds vbar in camera axes and featw[i] = clamp(rho, 0, 2)
//   tileinfo[i] = (x0 | y0 << 16, rect width | height << 16, fp32 bits of z, rect count)
//   counts[i]   = rect count (0 if culled)
//   dkeys[i], dvals[i] (optional) = (packed tile rect << 32 | fp32 bits of z, or 0xFFFFFFFF if culled), i
// Returns the low half of the depth-sort key: the fp32 bits of z, 0xFFFFFFFF if culled.
// PART: PRE_ALL -- everything. PRE_GEO -- what the list building needs (tile info, counts, depth pair) without the
// record: the 192 B of SH coefficients are not read (lazy lists: most Gaussians are never composited). Whether a
// Gaussian survives depends on its colour only through the non-finite-colour cull, which needs non-finite or
// astronomically large coefficients: relayout_kernel flags those Gaussians (shflag) and only they evaluate their
// colour here. PRE_REC -- recompute the same values and write the record only (shade_kernel).
enum { PRE_ALL = 0, PRE_GEO = 1, PRE_REC = 2 };
template <int PART>
__device__ __forceinline__ uint32_t
preprocess_point(const FrameParams& P, uint32_t n, uint32_t i, const uint8_t* __restrict__ shflag,
                 const float4* __restrict__ A0, const float4* __restrict__ A1,
                 const float4* __restrict__ A2, const float4* __restrict__ A3,
                 const float4* __restrict__ SH, float4* __restrict__ record,
                 uint4* __restrict__ tileinfo, uint32_t* __restrict__ counts,
                 uint64_t* __restrict__ dkeys, uint32_t* __restrict__ dvals, float* __restrict__ featw) {

  const float4 a0 = ldg_stream_f4(A0 + i);
  const float4 a1 = ldg_stream_f4(A1 + i);
  const float4 a2 = ldg_stream_f4(A2 + i);
  const float4 a3 = ldg_stream_f4(A3 + i);

  bool valid = true;
  float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0, r2 = r0;
  uint4 ti = make_uint4(0u, 0u, 0u, 0u);

  // P1: Eq. 6. sinpi gives an exact range reduction of 2 pi (t - tau) / l.
  const float dt = P.t - a0.w;
  const float m = P.linear ? dt : P.l_over_2pi * sinpif(P.two_over_l * dt);
  // staticness rho = beta / l; beta = +INF is rho = +INF whatever l
  const float rho = a1.w > 3.0e38f ? a1.w : a1.w * P.inv_l;
  // Eq. 12: temporal-smoothing state mu~(t1) + vbar dts, vbar = v exp(-rho/2) (Eq. 10)
  float mm = m;
  if (P.dts != 0.f) mm = fmaf(expf(-0.5f * rho), P.dts, m);
  const float wx = fmaf(mm, a1.x, a0.x), wy = fmaf(mm, a1.y, a0.y), wz = fmaf(mm, a1.z, a0.z);
  // P2: Eq. 7 (beta = +INF gives exp(-0) = 1)
  const float op = a3.w * expf(-0.5f * (dt * dt) / (a1.w * a1.w));
  // P3: opacity cull; the comparison is false for NaN
  valid = (op >= PVG_ALPHA_MIN) && (op <= 3.0e38f);
  // staticness filter: keep rho_min <= rho <= rho_max
  if (P.filter) valid = valid && (rho >= P.rho_min) && !(rho > P.rho_max);
  // P4: camera space + near cull
  const float px = fmaf(P.R[0], wx, fmaf(P.R[1], wy, fmaf(P.R[2], wz, P.T[0])));
  const float py = fmaf(P.R[3], wx, fmaf(P.R[4], wy, fmaf(P.R[5], wz, P.T[1])));
  const float pz = fmaf(P.R[6], wx, fmaf(P.R[7], wy, fmaf(P.R[8], wz, P.T[2])));
  valid = valid && (pz > P.znear) && (pz <= 3.0e38f) && (fabsf(px) <= 3.0e38f) && (fabsf(py) <= 3.0e38f);

  float mx = 0.f, my = 0.f, hx = 0.f, hy = 0.f;
  if (valid) {
    // P5: M = R(q) diag(s); Sigma = M M^T (never formed)
    const float qw = a2.x, qx = a2.y, qy = a2.z, qz = a2.w;
    const float R00 = 1.f - 2.f * (qy * qy + qz * qz), R01 = 2.f * (qx * qy - qw * qz), R02 = 2.f * (qx * qz + qw * qy);
    const float R10 = 2.f * (qx * qy + qw * qz), R11 = 1.f - 2.f * (qx * qx + qz * qz), R12 = 2.f * (qy * qz - qw * qx);
    const float R20 = 2.f * (qx * qz - qw * qy), R21 = 2.f * (qy * qz + qw * qx), R22 = 1.f - 2.f * (qx * qx + qy * qy);
    // P6: T = J W with the Jacobian guard (S15)
    const float iz = 1.0f / pz;
    const float xz = px / pz, yz = py / pz;
    const float tx = fminf(P.limx, fmaxf(-P.limx, xz));
    const float ty = fminf(P.limy, fmaxf(-P.limy, yz));
    const float j00 = P.fx * iz, j02 = -P.fx * tx * iz;  // -fx * xbar / z^2 with xbar = tx * z
    const float j11 = P.fy * iz, j12 = -P.fy * ty * iz;
    const float t00 = fmaf(j00, P.R[0], j02 * P.R[6]), t01 = fmaf(j00, P.R[1], j02 * P.R[7]), t02 = fmaf(j00, P.R[2], j02 * P.R[8]);
    const float t10 = fmaf(j11, P.R[3], j12 * P.R[6]), t11 = fmaf(j11, P.R[4], j12 * P.R[7]), t12 = fmaf(j11, P.R[5], j12 * P.R[8]);
    // U = T M (2x3); Sigma' = U U^T; det(U U^T) = |U0 x U1|^2 (Lagrange), free of the
    // cancellation in cxx*cyy - cxy^2
    const float u00 = (t00 * R00 + t01 * R10 + t02 * R20) * a3.x;
    const float u01 = (t00 * R01 + t01 * R11 + t02 * R21) * a3.y;
    const float u02 = (t00 * R02 + t01 * R12 + t02 * R22) * a3.z;
    const float u10 = (t10 * R00 + t11 * R10 + t12 * R20) * a3.x;
    const float u11 = (t10 * R01 + t11 * R11 + t12 * R21) * a3.y;
    const float u12 = (t10 * R02 + t11 * R12 + t12 * R22) * a3.z;
    const float sxx = u00 * u00 + u01 * u01 + u02 * u02;
    const float sxy = u00 * u10 + u01 * u11 + u02 * u12;
    const float syy = u10 * u10 + u11 * u11 + u12 * u12;
    const float c0 = u01 * u12 - u02 * u11, c1 = u02 * u10 - u00 * u12, c2 = u00 * u11 - u01 * u10;
    const float det0 = c0 * c0 + c1 * c1 + c2 * c2;
    const float cxx = sxx + PVG_DILATE, cyy = syy + PVG_DILATE;
    const float det = det0 + PVG_DILATE * (sxx + syy) + PVG_DILATE * PVG_DILATE;
    // P7: conic
    valid = (det > 0.f) && (det <= 3.0e38f);
    const float idet = 1.0f / det;
    const float ca = cyy * idet, cb = -sxy * idet, cc = cxx * idet;
    // P8, P9
    mx = fmaf(P.fx, xz, P.cx);
    my = fmaf(P.fy, yz, P.cy);
    const float kk = 2.0f * logf(255.0f * op);
    hx = sqrtf(kk * cxx);
    hy = sqrtf(kk * cyy);
    valid = valid && (fabsf(mx) <= 3.0e38f) && (fabsf(my) <= 3.0e38f) && (hx <= 3.0e38f) && (hy <= 3.0e38f);
    if (valid) {
      // P10: tile rectangle; the float->int decisions use individually rounded fp32 ops
      float x0 = __fmul_rn(__fsub_rn(mx, hx), 0.0625f), x1 = __fmul_rn(__fadd_rn(mx, hx), 0.0625f);
      float y0 = __fmul_rn(__fsub_rn(my, hy), 0.0625f), y1 = __fmul_rn(__fadd_rn(my, hy), 0.0625f);
      const float TXf = (float)P.tiles_x, TYf = (float)P.tiles_y;
      x0 = fminf(fmaxf(x0, -1.0f), TXf); x1 = fminf(fmaxf(x1, -1.0f), TXf);
      y0 = fminf(fmaxf(y0, -1.0f), TYf); y1 = fminf(fmaxf(y1, -1.0f), TYf);
      const int tx0 = max((int)floorf(x0), 0), tx1 = min((int)floorf(x1), P.tiles_x - 1);
      // the band of tile rows of this render: duplicate into own tiles only
      const int ty0 = max((int)floorf(y0), P.band_y0), ty1 = min((int)floorf(y1), P.band_y1 - 1);
      valid = (tx0 <= tx1) && (ty0 <= ty1);
      if (valid) {
        const uint32_t w = (uint32_t)(tx1 - tx0 + 1), h = (uint32_t)(ty1 - ty0 + 1);
        ti = make_uint4((uint32_t)tx0 | ((uint32_t)ty0 << 16), w | (h << 16), __float_as_uint(pz), w * h);
        r0 = make_float4(mx, my, pz, op);
        r1 = make_float4(ca, cb, cc, hx);
      }
    }
  }

  if (valid && P.target == 1) {
    // "Flexible rendering ... by replacing the color c in Eq. (3)" with the quantities of the
    // dynamic element analysis (L298): the average velocity vbar = v exp(-rho/2) (Eq. 10) in camera axes, and the
    // staticness clamped to [0, 2]. No SH read in this mode.
    const float e = expf(-0.5f * rho);
    const float vx = e * a1.x, vy = e * a1.y, vz = e * a1.z;
    r2 = make_float4(fmaf(P.R[0], vx, fmaf(P.R[1], vy, P.R[2] * vz)), fmaf(P.R[3], vx, fmaf(P.R[4], vy, P.R[5] * vz)),
                     fmaf(P.R[6], vx, fmaf(P.R[7], vy, P.R[8] * vz)), hy);
    if (PART != PRE_GEO) featw[i] = fminf(fmaxf(rho, 0.f), 2.0f);
    if (!((fabsf(r2.x) <= 3.0e38f) && (fabsf(r2.y) <= 3.0e38f) && (fabsf(r2.z) <= 3.0e38f))) {
      valid = false;
      r0 = make_float4(0.f, 0.f, 0.f, 0.f); r1 = r0; r2 = r0;
      ti = make_uint4(0u, 0u, 0u, 0u);
    }
  } else if (valid && (PART != PRE_GEO || shflag[i])) {
    // P11: SH colour; only survivors touch the 192 B of coefficients
    float dx = wx - P.campos[0], dy = wy - P.campos[1], dz = wz - P.campos[2];
    const float inv = 1.0f / sqrtf(dx * dx + dy * dy + dz * dz);
    dx *= inv; dy *= inv; dz *= inv;
    float f[48];
    const int nplanes = P.sh_degree == 0 ? 1 : (P.sh_degree == 1 ? 3 : (P.sh_degree == 2 ? 7 : 12));
#pragma unroll
    for (int p = 0; p < 12; ++p) {
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (p < nplanes) v = ldg_stream_f4(SH + (size_t)p * n + i);
      f[4 * p] = v.x; f[4 * p + 1] = v.y; f[4 * p + 2] = v.z; f[4 * p + 3] = v.w;
    }
    // coefficient k, channel ch = f[3k + ch]; zero the tail of the last plane past the degree
    const int nfl = 3 * (P.sh_degree + 1) * (P.sh_degree + 1);
#pragma unroll
    for (int k = 0; k < 48; ++k) if (k >= nfl) f[k] = 0.f;
    const float xx = dx * dx, yy = dy * dy, zz = dz * dz, xy = dx * dy, yz2 = dy * dz, xz2 = dx * dz;
    float Y[16];
    Y[0] = SH_C0;
    Y[1] = -SH_C1 * dy; Y[2] = SH_C1 * dz; Y[3] = -SH_C1 * dx;
    Y[4] = SH_C2A * xy; Y[5] = -SH_C2A * yz2; Y[6] = SH_C2B * (2.f * zz - xx - yy);
    Y[7] = -SH_C2A * xz2; Y[8] = SH_C2C * (xx - yy);
    Y[9] = -SH_C3A * dy * (3.f * xx - yy); Y[10] = SH_C3B * xy * dz;
    Y[11] = -SH_C3C * dy * (4.f * zz - xx - yy); Y[12] = SH_C3D * dz * (2.f * zz - 3.f * xx - 3.f * yy);
    Y[13] = -SH_C3C * dx * (4.f * zz - xx - yy); Y[14] = SH_C3E * dz * (xx - yy);
    Y[15] = -SH_C3A * dx * (xx - 3.f * yy);
    float cr = 0.5f, cg = 0.5f, cbl = 0.5f;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      cr = fmaf(Y[k], f[3 * k], cr);
      cg = fmaf(Y[k], f[3 * k + 1], cg);
      cbl = fmaf(Y[k], f[3 * k + 2], cbl);
    }
    cr = fmaxf(cr, 0.f); cg = fmaxf(cg, 0.f); cbl = fmaxf(cbl, 0.f);
    if ((cr <= 3.0e38f) && (cg <= 3.0e38f) && (cbl <= 3.0e38f)) {
      r2 = make_float4(cr, cg, cbl, hy);
    } else {  // non-finite colour never poisons the image
      valid = false;
      r0 = make_float4(0.f, 0.f, 0.f, 0.f); r1 = r0;
      ti = make_uint4(0u, 0u, 0u, 0u);
    }
  }

  if (PART != PRE_GEO) {
    record[3 * (size_t)i] = r0;
    record[3 * (size_t)i + 1] = r1;
    record[3 * (size_t)i + 2] = r2;
  }
  if (PART == PRE_REC) return valid ? ti.z : 0xFFFFFFFFu;
  tileinfo[i] = ti;
  counts[i] = ti.w;
  if (dkeys) {
    // upper half: (x0, y0, x1, y1) of the tile rectangle, 8 bits each -- payload that rides through the
    // depth sort, so the block-entry scan and emission read it sequentially instead of gathering tileinfo
    uint32_t rect = 0;
    if (P.pack_rect) {
      const uint32_t x0 = ti.x & 0xFFFFu, y0 = ti.x >> 16;
      rect = x0 | (y0 << 8) | ((x0 + (ti.y & 0xFFFFu) - 1u) << 16) | ((y0 + (ti.y >> 16) - 1u) << 24);
    }
    dkeys[i] = valid ? (((uint64_t)rect << 32) | ti.z) : 0xFFFFFFFFull;
    dvals[i] = i;
  }
  return valid ? ti.z : 0xFFFFFFFFu;
}

// PRE_CHUNKS consecutive groups of 256 Gaussians per CTA. With dhist != nullptr the CTA also counts the four
// 8-bit digits of its depth keys in shared memory, adds them to dhist[4][256] (zeroed) and the last CTA to
// finish (dhist[1024] counts them) turns the counts into the exclusive prefixes the onesweep passes of the
// depth sort start from -- the keys are in registers here; a histogram kernel would read them back from HBM.
#ifndef PVG_PRE_CHUNKS
#define PVG_PRE_CHUNKS 4
#endif
constexpr int PRE_CHUNKS = PVG_PRE_CHUNKS;
template <int PART>
__global__ void __launch_bounds__(256)
preprocess_kernel(const __grid_constant__ FrameParams P, uint32_t n, const uint8_t* __restrict__ shflag,
                  const float4* __restrict__ A0, const float4* __restrict__ A1,
                  const float4* __restrict__ A2, const float4* __restrict__ A3,
                  const float4* __restrict__ SH, float4* __restrict__ record,
                  uint4* __restrict__ tileinfo, uint32_t* __restrict__ counts,
                  uint64_t* __restrict__ dkeys, uint32_t* __restrict__ dvals, float* __restrict__ featw,
                  uint32_t* __restrict__ dhist) {
  __shared__ uint32_t s_hist[4 * 256];
  if (dhist) {
#pragma unroll
    for (int k = 0; k < 4; ++k) s_hist[k * 256 + threadIdx.x] = 0;
    __syncthreads();
  }
#pragma unroll 1
  for (int c = 0; c < PRE_CHUNKS; ++c) {
    const uint32_t i = (blockIdx.x * PRE_CHUNKS + c) * 256u + threadIdx.x;
    if (i >= n) break;
    const uint32_t z = preprocess_point<PART>(P, n, i, shflag, A0, A1, A2, A3, SH, record, tileinfo, counts, dkeys, dvals, featw);
    if (dhist) {
#pragma unroll
      for (int k = 0; k < 4; ++k) atomicAdd(&s_hist[k * 256 + ((z >> (8 * k)) & 0xFFu)], 1u);
    }
  }
  if (!dhist) return;
  __syncthreads();
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const uint32_t v = s_hist[k * 256 + threadIdx.x];
    if (v) atomicAdd(&dhist[k * 256 + threadIdx.x], v);
  }
  __shared__ bool s_last;
  __shared__ uint32_t s_warp[8];
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) s_last = atomicAdd(dhist + 1024, 1u) == gridDim.x - 1;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  for (int k = 0; k < 4; ++k) {
    const uint32_t v = __ldcg(dhist + k * 256 + threadIdx.x);
    uint32_t incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
      if (lane >= d) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    uint32_t wex = 0;
    for (uint32_t w = 0; w < warp; ++w) wex += s_warp[w];
    dhist[k * 256 + threadIdx.x] = wex + incl - v;
    __syncthreads();
  }
}

// The records PRE_GEO left out, for the Gaussians at depth ranks [*r_lo (or 0), *r_hi + 1 (or n)) of the sorted
// order: the same arithmetic as preprocess_kernel<PRE_ALL>, so the records are bit-identical to an eager frame.
// only_if: nothing to do when *only_if == 0 (lazy lists: the second round runs only if a tile was parked).
__global__ void __launch_bounds__(256)
shade_kernel(const __grid_constant__ FrameParams P, uint32_t n, const uint64_t* __restrict__ keys, const uint32_t* __restrict__ visit,
             const uint32_t* __restrict__ r_lo, const uint32_t* __restrict__ r_hi, const uint32_t* __restrict__ only_if,
             const float4* __restrict__ A0, const float4* __restrict__ A1, const float4* __restrict__ A2,
             const float4* __restrict__ A3, const float4* __restrict__ SH, float4* __restrict__ record, float* __restrict__ featw,
             int zero_culled /* pvg_debug_view: the culled Gaussians' records read as zero */) {
  if (only_if && *only_if == 0u) return;
  const uint32_t lo = r_lo ? *r_lo + 1u : 0u, hi = r_hi ? min(*r_hi + 1u, n) : n;
  const uint32_t r = lo + blockIdx.x * 256u + threadIdx.x;
  if (r >= hi) return;
  if ((uint32_t)keys[r] == 0xFFFFFFFFu) {   // culled (they sort last): nobody composites them
    if (zero_culled) {
      const size_t g = visit[r];
      record[3 * g] = record[3 * g + 1] = record[3 * g + 2] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    return;
  }
  preprocess_point<PRE_REC>(P, n, visit[r], nullptr, A0, A1, A2, A3, SH, record, nullptr, nullptr, nullptr, nullptr, featw);
}

// One-off re-layout of the caller's arrays into the SoA float4 model (pvg_create_scene).
__global__ void __launch_bounds__(256)
relayout_kernel(uint32_t n, const float* __restrict__ mu, const float* __restrict__ quat,
                const float* __restrict__ scale, const float* __restrict__ opacity,
                const float* __restrict__ sh, const float* __restrict__ tau,
                const float* __restrict__ beta, const float* __restrict__ vel,
                float4* __restrict__ A0, float4* __restrict__ A1, float4* __restrict__ A2,
                float4* __restrict__ A3, float4* __restrict__ SH, uint8_t* __restrict__ shflag) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  // shflag: could the colour 0.5 + sum Y_k f_k be non-finite? |Y_k| < 3, so not while the coefficients are finite
  // and their absolute sum stays below 1e37
  float asum = 0.f;
  for (int k = 0; k < 48; ++k) asum += fabsf(sh[48 * (size_t)i + k]);
  shflag[i] = (asum < 1.0e37f) ? 0 : 1;   // NaN and inf fail the comparison
  A0[i] = make_float4(mu[3 * (size_t)i], mu[3 * (size_t)i + 1], mu[3 * (size_t)i + 2], tau[i]);
  A1[i] = make_float4(vel[3 * (size_t)i], vel[3 * (size_t)i + 1], vel[3 * (size_t)i + 2], beta[i]);
  const float qw = quat[4 * (size_t)i], qx = quat[4 * (size_t)i + 1], qy = quat[4 * (size_t)i + 2], qz = quat[4 * (size_t)i + 3];
  const float qn = 1.0f / sqrtf(qw * qw + qx * qx + qy * qy + qz * qz);
  A2[i] = make_float4(qw * qn, qx * qn, qy * qn, qz * qn);
  A3[i] = make_float4(scale[3 * (size_t)i], scale[3 * (size_t)i + 1], scale[3 * (size_t)i + 2], opacity[i]);
  const float4* src = reinterpret_cast<const float4*>(sh + 48 * (size_t)i);  // 192 B rows: 16 B aligned
#pragma unroll
  for (int p = 0; p < 12; ++p) SH[(size_t)p * n + i] = src[p];
}

}  // namespace pvg

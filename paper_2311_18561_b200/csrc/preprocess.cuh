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
#include "onesweep.cuh"

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

// sin(pi x) in double, |error| < 1e-13: x is reduced to [-1, 1] by the nearest even integer (exact), folded to
// [-1/2, 1/2] by sin(pi (s - x)) = sin(pi x) for s = +-1 (exact), and summed as the odd Taylor polynomial of degree
// 17 (its remainder at 1/2 is 4e-14).
__device__ __forceinline__ double sinpi_reduced(double x) {
  x = fma(-2.0, rint(0.5 * x), x);
  if (fabs(x) > 0.5) x = copysign(1.0, x) - x;
  const double x2 = x * x;
  double p = 7.952054001475513e-07;
  p = fma(p, x2, -2.1915353447830217e-05);
  p = fma(p, x2, 0.00046630280576761255);
  p = fma(p, x2, -0.0073704309457143504);
  p = fma(p, x2, 0.08214588661112823);
  p = fma(p, x2, -0.5992645293207921);
  p = fma(p, x2, 2.5501640398773455);
  p = fma(p, x2, -5.16771278004997);
  p = fma(p, x2, 3.141592653589793);
  return p * x;
}

// Model layout in HBM (built once by relayout_kernel):
//   A0[i] = (mu.x, mu.y, mu.z, tau)     A1[i] = (v.x, v.y, v.z, beta)
//   A2[i] = quaternion (w,x,y,z) as given (normalised inside R(q))   A3[i] = (s.x, s.y, s.z, o)
//   SH[p][i], p = 0..11: floats 4p..4p+3 of the point's [16][3] coefficient block
// Outputs:
//   record[3 i + {0,1,2}] = (mx,my,z,o~), (a,b,c,hx), (r,g,b,hy)   -- all 0 if culled; with P.target == 1 the
//                           colour slot holds vbar in camera axes and featw[i] = clamp(rho, 0, 2)
//   tileinfo[i] = (x0 | y0 << 16, rect width | height << 16, fp32 bits of z, rect count)
//   counts[i]   = rect count (0 if culled)
//   dkeys[i] (optional) = (packed tile rect << 32 | depth key, or 0xFFFFFFFF if culled); the pair's value is i itself
//                           depth key = fp32 bits of z - fp32 bits of znear (z > znear > 0: positive, same order as z)
// Returns the depth key, 0xFFFFFFFF if culled.
// PART: PRE_ALL -- everything. PRE_GEO -- what the list building needs (tile info, counts, depth pair) without the
// record: the 192 B of SH coefficients are not read (lazy lists: most Gaussians are never composited). Whether a
// Gaussian survives depends on its colour only through the non-finite-colour cull, which needs non-finite or
// astronomically large coefficients: relayout_kernel flags those Gaussians (shflag) and only they evaluate their
// colour here. PRE_REC -- recompute the same values and write the record only (shade_kernel).
enum { PRE_ALL = 0, PRE_GEO = 1, PRE_REC = 2 };
template <int PART>
__device__ __forceinline__ uint64_t
preprocess_loaded(const FrameParams& P, uint32_t n, uint32_t i, const float4 a0, const float4 a1, const float4 a2, const float4 a3,
                  const bool shade_here, const float4* __restrict__ SH, float4* __restrict__ record,
                  uint4* __restrict__ tileinfo, uint32_t* __restrict__ counts,
                  uint64_t* __restrict__ dkeys, uint32_t* __restrict__ dvals, float* __restrict__ featw);
template <int PART>
__device__ __forceinline__ uint64_t
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
  // PRE_GEO: the colour flag is fetched with the model, not when the survivor is known -- a load issued that late is a
  // second DRAM round trip on every warp's path (ncu: as many stall samples as the four model loads together)
  const bool shade_here = PART != PRE_GEO || (shflag != nullptr && __ldg(shflag + i) != 0);
  return preprocess_loaded<PART>(P, n, i, a0, a1, a2, a3, shade_here, SH, record, tileinfo, counts, dkeys, dvals, featw);
}

template <int PART>
__device__ __forceinline__ uint64_t
preprocess_loaded(const FrameParams& P, uint32_t n, uint32_t i, const float4 a0, const float4 a1, const float4 a2, const float4 a3,
                  const bool shade_here, const float4* __restrict__ SH, float4* __restrict__ record,
                  uint4* __restrict__ tileinfo, uint32_t* __restrict__ counts,
                  uint64_t* __restrict__ dkeys, uint32_t* __restrict__ dvals, float* __restrict__ featw) {
  bool valid = true;
  float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0, r2 = r0;
  uint4 ti = make_uint4(0u, 0u, 0u, 0u);

  // P1, P4, P8 -- the chain mu~(t) -> p_cam -> (mx, my) -- run in DOUBLE. In fp32 the rounding of t - tau alone
  // (3e-8) moves a fast, near Gaussian (|v| = 20 m/s at z = 2 m, f = 2000 px) by 6e-4 px, and the three dot products
  // and the division of the projection add a few ulps of coordinates of up to 2000 px (1.2e-4 px each): together up
  // to 3e-4 px in the mean, which through d alpha / d mean <= 0.6 o~ / sigma was the whole end-to-end image error
  // (6e-4 against the oracle's own record). In double the record's (mx, my, z) are the
  // correctly rounded fp32 values of the exact ones. B200 issues FP64 at half the FP32 rate and this kernel is
  // HBM-bound; the chain is kept to ~45 double instructions (polynomial sine, Newton reciprocal).
  // P1: Eq. 6, sin(2 pi dt / l) = sin(pi x) with x = 2 dt / l reduced to [-1/2, 1/2] exactly.
  const double dtd = P.t1 - (double)a0.w;   // exact
  double md = dtd;
  if (!P.linear) md = P.l_over_2pi * sinpi_reduced(P.two_over_l * dtd);
  // staticness rho = beta / l; beta = +INF is rho = +INF whatever l
  const float rho = a1.w > 3.0e38f ? a1.w : a1.w * P.inv_l;
  // Eq. 12: temporal-smoothing state mu~(t1) + vbar dts, vbar = v exp(-rho/2) (Eq. 10)
  if (P.dts != 0.f) {
    const double rhod = a1.w > 3.0e38f ? (double)a1.w : (double)a1.w * P.inv_l_d;
    md = fma(exp(-0.5 * rhod), (double)P.dts, md);
  }
  const double wxd = fma(md, (double)a1.x, (double)a0.x), wyd = fma(md, (double)a1.y, (double)a0.y),
               wzd = fma(md, (double)a1.z, (double)a0.z);
  const float wx = (float)wxd, wy = (float)wyd, wz = (float)wzd;
  // P2: Eq. 7 (beta = +INF gives exp(-0) = 1), fp32 on the exact t - tau: the exponent of a survivor is above
  // ln(1/255) = -5.5, three roundings of it are 1e-6 absolute
  const float dtb = (float)dtd / a1.w;
  const float op = a3.w * expf(-0.5f * dtb * dtb);
  // P3: opacity cull; the comparison is false for NaN
  valid = (op >= PVG_ALPHA_MIN) && (op <= 3.0e38f);
  // staticness filter: keep rho_min <= rho <= rho_max
  if (P.filter) valid = valid && (rho >= P.rho_min) && !(rho > P.rho_max);
  // P4: camera space + near cull
  const double pxd = fma(P.Rd[0], wxd, fma(P.Rd[1], wyd, fma(P.Rd[2], wzd, P.Td[0])));
  const double pyd = fma(P.Rd[3], wxd, fma(P.Rd[4], wyd, fma(P.Rd[5], wzd, P.Td[1])));
  const double pzd = fma(P.Rd[6], wxd, fma(P.Rd[7], wyd, fma(P.Rd[8], wzd, P.Td[2])));
  const float px = (float)pxd, py = (float)pyd, pz = (float)pzd;
  valid = valid && (pz > P.znear) && (pz <= 3.0e38f) && (fabsf(px) <= 3.0e38f) && (fabsf(py) <= 3.0e38f);

  float mx = 0.f, my = 0.f, hx = 0.f, hy = 0.f;
  if (valid) {
    // P5: M = R(q) diag(s); Sigma = M M^T (never formed). q is stored as given: R(q / |q|) = I + (2 / |q|^2) (...)
    // needs no square root.
    const float qw = a2.x, qx = a2.y, qy = a2.z, qz = a2.w;
    const float q2 = 2.0f / (qw * qw + qx * qx + qy * qy + qz * qz);
    const float R00 = 1.f - q2 * (qy * qy + qz * qz), R01 = q2 * (qx * qy - qw * qz), R02 = q2 * (qx * qz + qw * qy);
    const float R10 = q2 * (qx * qy + qw * qz), R11 = 1.f - q2 * (qx * qx + qz * qz), R12 = q2 * (qy * qz - qw * qx);
    const float R20 = q2 * (qx * qz - qw * qy), R21 = q2 * (qy * qz + qw * qx), R22 = 1.f - q2 * (qx * qx + qy * qy);
    // P6: T = J W with the Jacobian guard (S15)
    const float iz = 1.0f / pz;
    // 1 / z in double from the fp32 reciprocal by two Newton steps (relative error 1e-7 -> 1e-14 -> 1e-28: rounding)
    double izd = (double)iz;
    izd = izd * fma(-pzd, izd, 2.0);
    izd = izd * fma(-pzd, izd, 2.0);
    const double xzd = pxd * izd, yzd = pyd * izd;
    const float xz = (float)xzd, yz = (float)yzd;
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
    const float syy = u10 * u10 + u11 * u11 + u12 * u12;
    const float c0 = u01 * u12 - u02 * u11, c1 = u02 * u10 - u00 * u12, c2 = u00 * u11 - u01 * u10;
    const float det0 = c0 * c0 + c1 * c1 + c2 * c2;
    const float cxx = sxx + PVG_DILATE, cyy = syy + PVG_DILATE;
    const float det = det0 + PVG_DILATE * (sxx + syy) + PVG_DILATE * PVG_DILATE;
    // P7: conic. The survival decision and the extents below use the fp32 covariance (the geometry pass and the
    // record pass must take them identically); the record's conic itself is computed in double (record passes only:
    // in the lazy mode ~12 % of the Gaussians): in fp32 U U^T loses C eps (f/z)^2 s_max^2 per entry -- for a needle
    // seen end-on a large multiple of the entry itself --, in double the conic is the correctly rounded one.
    valid = (det > 0.f) && (det <= 3.0e38f);
    float ca = 0.f, cb = 0.f, cc = 0.f;
    if (PART != PRE_GEO) {
      const double dqw = a2.x, dqx = a2.y, dqz = a2.w, dqy = a2.z;
      const double n2 = fma(dqw, dqw, fma(dqx, dqx, fma(dqy, dqy, dqz * dqz)));
      double s2 = (double)(1.0f / (float)n2);
      s2 = s2 * fma(-n2, s2, 2.0);
      s2 = s2 * fma(-n2, s2, 2.0);
      s2 += s2;   // 2 / |q|^2
      const double D00 = fma(-s2, fma(dqy, dqy, dqz * dqz), 1.0), D01 = s2 * fma(dqx, dqy, -dqw * dqz), D02 = s2 * fma(dqx, dqz, dqw * dqy);
      const double D10 = s2 * fma(dqx, dqy, dqw * dqz), D11 = fma(-s2, fma(dqx, dqx, dqz * dqz), 1.0), D12 = s2 * fma(dqy, dqz, -dqw * dqx);
      const double D20 = s2 * fma(dqx, dqz, -dqw * dqy), D21 = s2 * fma(dqy, dqz, dqw * dqx), D22 = fma(-s2, fma(dqx, dqx, dqy * dqy), 1.0);
      const double txd = fmin(P.limxd, fmax(-P.limxd, xzd)), tyd = fmin(P.limyd, fmax(-P.limyd, yzd));
      const double e00 = P.fxd * izd, e02 = -e00 * txd, e11 = P.fyd * izd, e12 = -e11 * tyd;
      const double T00 = fma(e00, P.Rd[0], e02 * P.Rd[6]), T01 = fma(e00, P.Rd[1], e02 * P.Rd[7]), T02 = fma(e00, P.Rd[2], e02 * P.Rd[8]);
      const double T10 = fma(e11, P.Rd[3], e12 * P.Rd[6]), T11 = fma(e11, P.Rd[4], e12 * P.Rd[7]), T12 = fma(e11, P.Rd[5], e12 * P.Rd[8]);
      const double sx = a3.x, sy = a3.y, sz = a3.z;
      const double U00 = fma(T00, D00, fma(T01, D10, T02 * D20)) * sx, U01 = fma(T00, D01, fma(T01, D11, T02 * D21)) * sy,
                   U02 = fma(T00, D02, fma(T01, D12, T02 * D22)) * sz;
      const double U10 = fma(T10, D00, fma(T11, D10, T12 * D20)) * sx, U11 = fma(T10, D01, fma(T11, D11, T12 * D21)) * sy,
                   U12 = fma(T10, D02, fma(T11, D12, T12 * D22)) * sz;
      const double Sxx = fma(U00, U00, fma(U01, U01, U02 * U02)) + (double)PVG_DILATE_D;
      const double Sxy = fma(U00, U10, fma(U01, U11, U02 * U12));
      const double Syy = fma(U10, U10, fma(U11, U11, U12 * U12)) + (double)PVG_DILATE_D;
      const double detd = fma(Sxx, Syy, -Sxy * Sxy);
      double idd = (double)(1.0f / (float)detd);
      idd = idd * fma(-detd, idd, 2.0);
      idd = idd * fma(-detd, idd, 2.0);
      ca = (float)(Syy * idd);
      cb = (float)(-Sxy * idd);
      cc = (float)(Sxx * idd);
    }
    // P8, P9
    mx = (float)fma(P.fxd, xzd, P.cxd);
    my = (float)fma(P.fyd, yzd, P.cyd);
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
  } else if (valid && shade_here) {
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
  if (PART == PRE_REC) return valid ? (uint64_t)ti.z : 0xFFFFFFFFull;
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
    const uint64_t key = valid ? (((uint64_t)rect << 32) | (ti.z - __float_as_uint(P.znear))) : 0xFFFFFFFFull;
    dkeys[i] = key;
    (void)dvals;   // the value of pair i is i: the first pass of the depth sort forms it instead of loading it
    return key;
  }
  return valid ? (uint64_t)(ti.z - __float_as_uint(P.znear)) : 0xFFFFFFFFull;
}

// PRE_CHUNKS consecutive groups of 256 Gaussians per CTA. With dhist != nullptr the CTA also counts the four digits
// (9 + 9 + 9 + 4 bits, onesweep.cuh "depth sort") of its survivors' depth keys in shared memory, adds them to
// dhist[4][512] (zeroed) and the last CTA to finish (dhist[DH_COUNTER] counts them) turns the counts into the
// exclusive prefixes the passes of the depth sort start from, and writes the sort's control block: the number of
// survivors S, which passes are the identity (one non-empty bin) and which buffer each pass reads -- the keys are in
// registers here; a histogram kernel would read them back from HBM.
// (B200, config 3, with the colour flag loaded up front: 4 chunks 0.0715 ms, 6: 0.0722, 8: 0.0709; with the next chunk's
// model lines prefetched into L2 while the current one is computed: 6: 0.0698, 8: 0.0687, 12: 0.0690. A register
// pipeline of the next chunk's values needs 80 registers, three CTAs per SM instead of four: 0.080.)
#ifndef PVG_PRE_CHUNKS
#define PVG_PRE_CHUNKS 8
#endif
#ifndef PVG_PRE_PF
#define PVG_PRE_PF 1
#endif

constexpr int PRE_CHUNKS = PVG_PRE_CHUNKS;

// FRONT (lazy lists with the front-first depth order, onesweep.cuh): instead of the digits the CTA counts, per bucket
// of the top key bits (key >> FR_SHIFT), its survivors and their block entries, and sums their tile instances; the last
// CTA picks the key threshold below which the first slab's owners lie (FrontCtl) and hands the frame's totals to the
// host: M, Mb, S, F -- all the host waits for.
// The geometry-only pass at 6 CTAs per SM (40 registers, 180 bytes of spills) instead of the 4 (64 registers) the compiler
// picks on its own: config 3 frame 0.2890 -> 0.2842 ms, config 4 0.6395 -> 0.6310 (5 CTAs: 0.2845; 7 and 8: 0.310 -- 32
// registers, 340 bytes of spills). The full pass (records with SH colour) keeps the compiler's choice (0: no minimum).
#ifndef PVG_PRE_MINB
#define PVG_PRE_MINB 6
#endif
template <int PART, bool FRONT>
__global__ void __launch_bounds__(256, PART == PRE_GEO ? PVG_PRE_MINB : 0)
preprocess_kernel(const __grid_constant__ FrameParams P, uint32_t n, const uint8_t* __restrict__ shflag,
                  const float4* __restrict__ A0, const float4* __restrict__ A1,
                  const float4* __restrict__ A2, const float4* __restrict__ A3,
                  const float4* __restrict__ SH, float4* __restrict__ record,
                  uint4* __restrict__ tileinfo, uint32_t* __restrict__ counts,
                  uint64_t* __restrict__ dkeys, uint32_t* __restrict__ dvals, float* __restrict__ featw,
                  uint32_t* __restrict__ dhist, volatile uint64_t* __restrict__ host_words /* mapped: [4] = S, [5] = final side, [6] = skipped passes (bit p); FRONT: [0] = M, [1] = Mb, [4] = S, [8] = F, [9] = top-digit flags */) {
  __shared__ uint32_t s_hist[DS_PASSES * DS_RADIX];
  static_assert(2 * FR_BUCKETS == DS_PASSES * DS_RADIX, "the bucket histograms reuse the digit histograms' words");
  if (dhist) {
#pragma unroll
    for (int k = 0; k < DS_PASSES * DS_RADIX / 256; ++k) s_hist[k * 256 + threadIdx.x] = 0;
    __syncthreads();
  }
  uint32_t inst = 0;   // FRONT: tile instances of this thread's survivors
#pragma unroll 1
  for (int c = 0; c < PRE_CHUNKS; ++c) {
    const uint32_t i = (blockIdx.x * PRE_CHUNKS + c) * 256u + threadIdx.x;
    if (i >= n) break;
#if PVG_PRE_PF
    if (c + 1 < PRE_CHUNKS && i + 256u < n) {
      asm volatile("prefetch.global.L2 [%0];" ::"l"(A0 + i + 256));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(A1 + i + 256));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(A2 + i + 256));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(A3 + i + 256));
    }
#endif
    const uint64_t key = preprocess_point<PART>(P, n, i, shflag, A0, A1, A2, A3, SH, record, tileinfo, counts, dkeys, dvals, featw);
    const uint32_t z = (uint32_t)key;
    if (dhist && z != 0xFFFFFFFFu) {
      if (FRONT) {
        const uint32_t r = (uint32_t)(key >> 32);
        const uint32_t x0 = r & 0xFFu, y0 = (r >> 8) & 0xFFu, x1 = (r >> 16) & 0xFFu, y1 = r >> 24;
        const uint32_t b = min(z >> FR_SHIFT, (uint32_t)FR_BUCKETS - 1u);
        atomicAdd(&s_hist[b], 1u);
        atomicAdd(&s_hist[FR_BUCKETS + b], ((x1 >> 3) - (x0 >> 3) + 1u) * ((y1 >> 3) - (y0 >> 3) + 1u));
        inst += (x1 - x0 + 1u) * (y1 - y0 + 1u);
      } else {
#pragma unroll
        for (int k = 0; k < DS_PASSES; ++k) atomicAdd(&s_hist[k * DS_RADIX + ((z >> ds_shift(k)) & ((1u << ds_bits(k)) - 1u))], 1u);
      }
    }
  }
  if (!dhist) return;
  __syncthreads();
#pragma unroll
  for (int k = 0; k < DS_PASSES * DS_RADIX / 256; ++k) {
    const uint32_t v = s_hist[k * 256 + threadIdx.x];
    if (v) atomicAdd(&dhist[k * 256 + threadIdx.x], v);
  }
  __shared__ bool s_last;
  __shared__ uint32_t s_warp[8], s_bins[8];
  if (FRONT) {
    inst = __reduce_add_sync(0xffffffffu, inst);   // < 2^32: 32 Gaussians of at most 2^16 tiles each
    if ((threadIdx.x & 31u) == 0 && inst) atomicAdd(reinterpret_cast<unsigned long long*>(dhist + DH_COUNTER + 2), (unsigned long long)inst);
  }
  // release: the barrier orders every thread's histogram atomics before thread 0, whose (cumulative) fence orders them
  // before its count -- one fence per CTA instead of one per thread (ncu: 1.1 stall cycles per issued instruction)
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    s_last = atomicAdd(dhist + DH_COUNTER, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  if (FRONT) {
    // thread t owns buckets 4 t .. 4 t + 3; inclusive sums of the survivors and of their block entries over the buckets
    __shared__ unsigned long long s_ent[8];
    uint32_t c[4], e[4];
    uint32_t csum = 0;
    unsigned long long esum = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      c[k] = __ldcg(dhist + 4 * threadIdx.x + k);
      e[k] = __ldcg(dhist + FR_BUCKETS + 4 * threadIdx.x + k);
      csum += c[k]; esum += e[k];
    }
    uint32_t cin = csum;
    unsigned long long ein = esum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t tc = __shfl_up_sync(0xffffffffu, cin, d);
      const unsigned long long te = __shfl_up_sync(0xffffffffu, ein, d);
      if (lane >= d) { cin += tc; ein += te; }
    }
    if (lane == 31) { s_warp[warp] = cin; s_ent[warp] = ein; }
    __syncthreads();
    uint32_t cex = 0, S = 0;
    unsigned long long eex = 0, Mb = 0;
    for (uint32_t w = 0; w < 8; ++w) {
      if (w < warp) { cex += s_warp[w]; eex += s_ent[w]; }
      S += s_warp[w]; Mb += s_ent[w];
    }
    cex += cin - csum; eex += ein - esum;   // exclusive of this thread's four buckets
    // the first slab: bin_emit's first launch forms the entries [0, emit_first * BF_TILE), and shade_kernel asks for
    // the owner of entry emit_first * BF_TILE: the front must hold more entries than that
    const unsigned long long target = ((unsigned long long)lazy_emit_first(Mb, P.lazy_slab, P.lazy_min_tiles) + 1ull) * (unsigned long long)PVG_EMIT_TILE;
    __shared__ uint32_t s_thr, s_front;
    if (threadIdx.x == 0) { s_thr = 0xFFFFFFFFu; s_front = S; }
    __syncthreads();
    if (Mb > target) {
      // the one bucket at which the inclusive entry sum first reaches the target
      unsigned long long run = eex;
      uint32_t crun = cex;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const unsigned long long before = run;
        run += e[k]; crun += c[k];
        const uint32_t b = 4 * threadIdx.x + k;
        if (before < target && run >= target && b + 1 < (uint32_t)FR_TOP) { s_thr = (b + 1u) << FR_SHIFT; s_front = crun; }
      }
    }
    // keys of 2^27 and beyond (buckets FR_TOP ..): which class has them decides its top-digit pass
    uint32_t far = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) if (4 * threadIdx.x + k >= (uint32_t)FR_TOP) far += c[k];
    far = __syncthreads_or(far != 0u);
    if (threadIdx.x == 0) {
      FrontCtl* fc = reinterpret_cast<FrontCtl*>(dhist + DH_CTL);
      const uint32_t thr = s_thr, F = s_front;
      fc->survivors = S; fc->front = F; fc->thr = thr;
      fc->top_front = (thr == 0xFFFFFFFFu && far) ? 1u : 0u;
      fc->top_back = (thr != 0xFFFFFFFFu && far) ? 1u : 0u;
      const unsigned long long M = *reinterpret_cast<const volatile unsigned long long*>(dhist + DH_COUNTER + 2);
      if (host_words) {
        host_words[0] = M; host_words[1] = Mb; host_words[4] = S; host_words[8] = F;
        host_words[9] = fc->top_front | (fc->top_back << 1);
      }
    }
    return;
  }
  uint32_t nonempty[DS_PASSES], total = 0;
  for (int k = 0; k < DS_PASSES; ++k) {
    // thread t owns bins 2 t, 2 t + 1 of the digit's 512
    const uint32_t v0 = __ldcg(dhist + k * DS_RADIX + 2 * threadIdx.x), v1 = __ldcg(dhist + k * DS_RADIX + 2 * threadIdx.x + 1);
    const uint32_t v = v0 + v1;
    uint32_t incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
      if (lane >= d) incl += t;
    }
    const uint32_t ne = __reduce_add_sync(0xffffffffu, (v0 ? 1u : 0u) + (v1 ? 1u : 0u));
    if (lane == 31) { s_warp[warp] = incl; s_bins[warp] = ne; }
    __syncthreads();
    uint32_t wex = 0, bins = 0, all = 0;
    for (uint32_t w = 0; w < 8; ++w) {
      if (w < warp) wex += s_warp[w];
      all += s_warp[w];
      bins += s_bins[w];
    }
    const uint32_t ex = wex + incl - v;
    dhist[k * DS_RADIX + 2 * threadIdx.x] = ex;
    dhist[k * DS_RADIX + 2 * threadIdx.x + 1] = ex + v0;
    nonempty[k] = bins;
    total = all;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    DepthCtl* ctl = reinterpret_cast<DepthCtl*>(dhist + DH_CTL);
    ctl->survivors = total;
    uint32_t side = 0;
    for (int k = 0; k < DS_PASSES; ++k) {
      const uint32_t skip = (k > 0 && nonempty[k] <= 1u) ? 1u : 0u;   // pass 0 always runs: it drops the culled pairs
      ctl->skip[k] = skip;
      ctl->in_side[k] = side;
      side ^= skip ^ 1u;
    }
    ctl->final_side = side;
    if (host_words) {
      uint32_t skips = 0;
      for (int k = 0; k < DS_PASSES; ++k) skips |= ctl->skip[k] << k;
      host_words[4] = total; host_words[5] = side; host_words[6] = skips;
    }
  }
}

// The records PRE_GEO left out, for the survivors at depth ranks [*r_lo + 1 (or 0), *r_hi + 1 (or nv)) of the sorted
// order (nv = S survivors): the same arithmetic as preprocess_kernel<PRE_ALL>, so the records are bit-identical to an
// eager frame. only_if: nothing to do when *only_if == 0 (lazy lists: the second round runs only if a tile was parked).
__global__ void __launch_bounds__(256)
shade_kernel(const __grid_constant__ FrameParams P, uint32_t n, uint32_t nv, const uint32_t* __restrict__ visit,
             const uint32_t* __restrict__ r_lo, const uint32_t* __restrict__ r_hi, const uint32_t* __restrict__ only_if,
             const float4* __restrict__ A0, const float4* __restrict__ A1, const float4* __restrict__ A2,
             const float4* __restrict__ A3, const float4* __restrict__ SH, float4* __restrict__ record, float* __restrict__ featw) {
  if (only_if && *only_if == 0u) return;
  const uint32_t lo = r_lo ? *r_lo + 1u : 0u, hi = r_hi ? min(*r_hi + 1u, nv) : nv;
  const uint32_t r = lo + blockIdx.x * 256u + threadIdx.x;
  if (r >= hi) return;
  preprocess_point<PRE_REC>(P, n, visit[r], nullptr, A0, A1, A2, A3, SH, record, nullptr, nullptr, nullptr, nullptr, featw);
}

// The records of the Gaussians in a device-side list (front-first depth order: the front, as depth_select_kernel
// compacted it -- in index order, before it is sorted: the records do not depend on the order, so this runs beside
// the sort on a stream of its own). *count entries; grid-stride, the launch does not know the count.
__global__ void __launch_bounds__(256)
shade_list_kernel(const __grid_constant__ FrameParams P, uint32_t n, const uint32_t* __restrict__ count, const uint32_t* __restrict__ list,
                  const float4* __restrict__ A0, const float4* __restrict__ A1, const float4* __restrict__ A2,
                  const float4* __restrict__ A3, const float4* __restrict__ SH, float4* __restrict__ record, float* __restrict__ featw) {
  const uint32_t c = *count;
  for (uint32_t r = blockIdx.x * 256u + threadIdx.x; r < c; r += gridDim.x * 256u)
    preprocess_point<PRE_REC>(P, n, list[r], nullptr, A0, A1, A2, A3, SH, record, nullptr, nullptr, nullptr, nullptr, featw);
}

// The records of ALL Gaussians in index order (coalesced model reads: 4 x faster than the gather by depth rank when
// most of the scene has to be shaded anyway -- the second round of a frame whose tiles parked, pvg_debug_view):
// survivors (counts[i] != 0) get their record, culled Gaussians zeros.
__global__ void __launch_bounds__(256)
shade_all_kernel(const __grid_constant__ FrameParams P, uint32_t n, const uint32_t* __restrict__ counts, const uint32_t* __restrict__ only_if,
                 const float4* __restrict__ A0, const float4* __restrict__ A1, const float4* __restrict__ A2,
                 const float4* __restrict__ A3, const float4* __restrict__ SH, float4* __restrict__ record, float* __restrict__ featw) {
  pdl_launch_dependents();
  pdl_wait();
  if (only_if && *only_if == 0u) return;
  // grid-stride: the launch that finds nothing to do (no tile parked) should cost a few hundred CTAs, not n / 256
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n; i += gridDim.x * 256u) {
    if (counts[i] == 0u) {
      record[3 * (size_t)i] = record[3 * (size_t)i + 1] = record[3 * (size_t)i + 2] = make_float4(0.f, 0.f, 0.f, 0.f);
      continue;
    }
    preprocess_point<PRE_REC>(P, n, i, nullptr, A0, A1, A2, A3, SH, record, nullptr, nullptr, nullptr, nullptr, featw);
  }
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
  A2[i] = make_float4(qw, qx, qy, qz);
  A3[i] = make_float4(scale[3 * (size_t)i], scale[3 * (size_t)i + 1], scale[3 * (size_t)i + 2], opacity[i]);
  const float4* src = reinterpret_cast<const float4*>(sh + 48 * (size_t)i);  // 192 B rows: 16 B aligned
#pragma unroll
  for (int p = 0; p < 12; ++p) SH[(size_t)p * n + i] = src[p];
}

}  // namespace pvg

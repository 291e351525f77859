// pvg_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct CPU oracle for the time-conditioned forward
// splatting render of "Periodic Vibration Gaussian" (arxiv 2311.18561),
// written from /root/reference/PAPER.md. It shares no code with the CUDA path
// (paper_2311_18561_b200/csrc) and may be imported only by tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg.
//
// Citations are PAPER.md:L<line> + equation; "S<n>"/"P<n>" are the readings of
// the silent points listed in DESIGN.md (taken from SURVEY.md section 8(c)).
//
// Floating point: Oracle-P and Oracle-R compute in double. The integer chain
// (tile rectangles, keys, sort, ranges) is defined on fp32 record values and
// takes its float->int decisions in fp32 (the kernel's precision), so that both
// sides decide from identical inputs in identical precision. Compile with
// -ffp-contract=off and without fast-math.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): closed forms T1..T8 of the
// paper, single-Gaussian image, stop/clamp/cutoff rules, brute force == binned,
// std::stable_sort equivalence on tiny scenes; for oracle_preprocess_state (Eq. 10 / 12,
// staticness filter) TestTemporalSmoothingState; for the sky cube map (oracle_sky_*) TestSky; for
// oracle_dynamics TestDynamicsTarget.
// "Absolute values on real data"
// is parity unpinned (the paper prints no worked numeric example).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr int kTile = 16;                   // S8: 16x16 tiles
constexpr double kAlphaMin = 1.0 / 255.0;   // S9: alpha cutoff
constexpr double kAlphaMax = 0.99;          // S9: alpha clamp
constexpr double kTStop = 1e-4;             // S9: transmittance stop
constexpr double kDilate = 0.3;             // S6: low-pass dilation (px^2)

struct Cam {
  int width, height;
  double fx, fy, cx, cy;
  double w2c[12];   // row-major 3x4 [R|T]
  double znear;
  double bg[3];
};

// slots of the wide double record (one row per Gaussian)
enum Slot {
  S_MU = 0,        // 0..2   mu~(t)                  Eq. 6
  S_OP = 3,        // o~(t)                          Eq. 7
  S_PCAM = 4,      // 4..6   camera-space position   P4
  S_SIG = 7,       // 7..12  Sigma xx xy xz yy yz zz P5
  S_COV = 13,      // 13..15 Sigma' xx xy yy (dilated) P6
  S_CONIC = 16,    // 16..18 a b c                   P7
  S_MEAN = 19,     // 19..20 mx my                   P8
  S_EXT = 21,      // 21..22 hx hy                   P9
  S_RGB = 23,      // 23..25 colour                  P11
  S_CULL = 26,     // 0 valid, 1 opacity, 2 near, 3 det, 4 rect, 5 non-finite
  S_RECT = 27,     // 27..30 tx0 ty0 tx1 ty1 (inclusive)
  S_COUNT = 31,
  S_STRIDE = 32
};

inline bool finite3(const double* p) {
  return std::isfinite(p[0]) && std::isfinite(p[1]) && std::isfinite(p[2]);
}

// Real spherical-harmonic basis to degree 3, closed forms, every constant from
// pi (P11 / S3). d must be a unit vector.
void sh_basis(const double d[3], double Y[16]) {
  const double x = d[0], y = d[1], z = d[2];
  const double xx = x * x, yy = y * y, zz = z * z;
  Y[0] = std::sqrt(1.0 / (4.0 * kPi));
  const double c1 = std::sqrt(3.0 / (4.0 * kPi));
  Y[1] = -c1 * y;
  Y[2] = c1 * z;
  Y[3] = -c1 * x;
  const double c2a = std::sqrt(15.0 / (4.0 * kPi));
  Y[4] = c2a * x * y;
  Y[5] = -c2a * y * z;
  Y[6] = std::sqrt(5.0 / (16.0 * kPi)) * (2.0 * zz - xx - yy);
  Y[7] = -c2a * x * z;
  Y[8] = std::sqrt(15.0 / (16.0 * kPi)) * (xx - yy);
  const double c3a = std::sqrt(35.0 / (32.0 * kPi));
  const double c3b = std::sqrt(21.0 / (32.0 * kPi));
  Y[9] = -c3a * y * (3.0 * xx - yy);
  Y[10] = std::sqrt(105.0 / (4.0 * kPi)) * x * y * z;
  Y[11] = -c3b * y * (4.0 * zz - xx - yy);
  Y[12] = std::sqrt(7.0 / (16.0 * kPi)) * z * (2.0 * zz - 3.0 * xx - 3.0 * yy);
  Y[13] = -c3b * x * (4.0 * zz - xx - yy);
  Y[14] = std::sqrt(105.0 / (16.0 * kPi)) * z * (xx - yy);
  Y[15] = -c3a * x * (xx - 3.0 * yy);
}

inline uint32_t f32_bits(float f) {
  uint32_t u;
  std::memcpy(&u, &f, 4);
  return u;
}

// Tile rectangle of one fp32 record row (P10), decisions taken in fp32.
// rec row = (mx,my,z,op, a,b,c,hx, r,g,b,hy). Returns count (0 if culled/empty).
inline uint32_t rect_of(const float* r, int TX, int TY, int rect[4]) {
  rect[0] = rect[1] = 0;
  rect[2] = rect[3] = -1;
  if (!(r[3] > 0.0f)) return 0;
  const float mx = r[0], my = r[1], hx = r[7], hy = r[11];
  float x0 = (mx - hx) * 0.0625f, x1 = (mx + hx) * 0.0625f;
  float y0 = (my - hy) * 0.0625f, y1 = (my + hy) * 0.0625f;
  x0 = std::fmin(std::fmax(x0, -1.0f), (float)TX);
  x1 = std::fmin(std::fmax(x1, -1.0f), (float)TX);
  y0 = std::fmin(std::fmax(y0, -1.0f), (float)TY);
  y1 = std::fmin(std::fmax(y1, -1.0f), (float)TY);
  int tx0 = (int)std::floor(x0), tx1 = (int)std::floor(x1);
  int ty0 = (int)std::floor(y0), ty1 = (int)std::floor(y1);
  tx0 = std::max(tx0, 0);
  ty0 = std::max(ty0, 0);
  tx1 = std::min(tx1, TX - 1);
  ty1 = std::min(ty1, TY - 1);
  if (tx0 > tx1 || ty0 > ty1) return 0;
  rect[0] = tx0; rect[1] = ty0; rect[2] = tx1; rect[3] = ty1;
  return (uint32_t)(tx1 - tx0 + 1) * (uint32_t)(ty1 - ty0 + 1);
}

// P13: which tiles of its rectangle can a Gaussian reach at all?
// The rectangle (P10) is the bounding box of the region R = { x : alpha(x) >= 1/255 } = { d : a dx^2 + 2 b dx dy + c dy^2
// <= k }, k = 2 ln(255 o~); towards its corners it holds tiles R does not touch. A tile is KEPT iff the box of its pixel
// centres, [16 tx + 0.5, 16 tx + 15.5] x [16 ty + 0.5, 16 ty + 15.5], intersects a slightly enlarged R. For one tile row
// (a band of dy) the x-projection of R within the band is an interval: its right end is the ellipse's right boundary
// xr(dy) = (-b dy + sqrt(a k - det dy^2)) / a at the dy of the band closest to where xr peaks (dy = -(b/c) dxm, dxm =
// sqrt(k c / det) the half-width of R), and mirrored for the left end. The decision is integer work: like P10 it is
// taken in fp32 from the fp32 record by INDIVIDUALLY ROUNDED operations (+, -, *, /, sqrt, min, max, floor, ceil), so
// that the CUDA path and this oracle decide identically. k is recovered without a logarithm from the record's
// extent, hx^2 = k Sigma'xx = k c / det. Margins (k (1 + 2e-4) + 2e-5, 1e-3 px) keep the test on the safe side of every
// rounding: a dropped tile has no pixel centre with alpha >= 1/255 (pinned by brute force in double).
struct ExactTile {
  bool refine;   // false: keep the whole rectangle (degenerate or non-finite conic)
  float mx, my, a, b, det, akk, dyr, ia;
};
inline ExactTile exact_tile_params(const float* r) {
  ExactTile e{};
  const float a = r[4], b = r[5], c = r[6], hx = r[7];
  const float det = a * c - b * b;
  const float k = ((hx * hx) * det) / c;
  const float kk = k * 1.0002f + 2e-5f;
  const float dxm = std::sqrt((kk * c) / det);
  const float dyr = -((b / c) * dxm);
  const float ia = 1.0f / a;
  e.mx = r[0]; e.my = r[1]; e.a = a; e.b = b; e.det = det; e.akk = a * kk; e.dyr = dyr; e.ia = ia;
  const float big = 3.0e38f;   // "finite" as the kernels test it: |x| <= 3e38 (false for NaN)
  e.refine = (det > 0.0f) && (a > 0.0f) && (c > 0.0f) && (std::fabs(kk) <= big) && (std::fabs(dxm) <= big) &&
             (std::fabs(ia) <= big) && (std::fabs(dyr) <= big) && (kk > 0.0f);
  return e;
}
// kept tiles [lo, hi] of tile row ty inside the rectangle's columns [tx0, tx1] (empty if lo > hi)
inline void exact_row_span(const ExactTile& e, int ty, int tx0, int tx1, int& lo, int& hi) {
  lo = tx0; hi = tx1;
  if (!e.refine) return;
  const float y0 = ((float)(16 * ty) + 0.5f) - e.my, y1 = y0 + 15.0f;
  // the band of pixel-centre rows lies wholly above or below R (|dy| > sqrt(a k / det) on its near side): no tile
  if ((y0 > 0.0f && e.akk - (e.det * y0) * y0 < 0.0f) || (y1 < 0.0f && e.akk - (e.det * y1) * y1 < 0.0f)) {
    hi = tx0 - 1;
    return;
  }
  const float tr = std::fmin(std::fmax(e.dyr, y0), y1);      // where the right boundary peaks inside the band
  const float tl = std::fmin(std::fmax(-e.dyr, y0), y1);     // and the left one
  const float dr = std::fmax(e.akk - (e.det * tr) * tr, 0.0f);
  const float dl = std::fmax(e.akk - (e.det * tl) * tl, 0.0f);
  const float xr = (std::sqrt(dr) - e.b * tr) * e.ia;
  const float xl = (-std::sqrt(dl) - e.b * tl) * e.ia;
  const float XR = (e.mx + xr) + 1e-3f, XL = (e.mx + xl) - 1e-3f;
  if (!(std::fabs(XR) <= 3.0e38f) || !(std::fabs(XL) <= 3.0e38f)) return;
  const float fh = std::floor((XR - 0.5f) * 0.0625f), fl = std::ceil((XL - 15.5f) * 0.0625f);
  // clamp in float before the conversion (|values| may exceed the int range)
  const int h = (int)std::fmin(std::fmax(fh, -2.0f), 1.0e6f), l = (int)std::fmin(std::fmax(fl, -2.0f), 1.0e6f);
  if (l > lo) lo = l;
  if (h < hi) hi = h;
}

// Depth order shared by every pixel (S11): ascending
// (fp32 bit pattern of z, Gaussian index) over the non-culled rows.
std::vector<uint32_t> depth_order(uint64_t n, const float* rec) {
  std::vector<uint32_t> ord;
  ord.reserve(n);
  for (uint64_t i = 0; i < n; ++i)
    if (rec[i * 12 + 3] > 0.0f) ord.push_back((uint32_t)i);
  std::stable_sort(ord.begin(), ord.end(), [&](uint32_t a, uint32_t b) {
    return f32_bits(rec[(uint64_t)a * 12 + 2]) < f32_bits(rec[(uint64_t)b * 12 + 2]);
  });
  return ord;
}

struct PixelOut {
  double rgb[3], depth, alpha, budget, cond, derived;
  uint64_t visited, contributed;
};

// End-to-end comparison: the image of ANOTHER fp32 record of the same scene (the CUDA
// path's own a1 output) is compared with the image of this record. Per Gaussian the caller states how far that
// other record may lie from this one -- slack[g] = { d mx, d my [px], d conic [absolute, each of a, b, c],
// d ln o~ [relative], d colour [absolute], d z [fp32 ulps] } -- and composite_pixel turns the statement into a per-pixel allowance
// by first-order propagation through Eq. 3:
//   d w      = |dw/dmx| d mx + |dw/dmy| d my + (dx^2/2 + dy^2/2 + |dx dy|) d conic + d ln o~     (w = ln alpha)
//   |dC/d alpha_i| <= T_i c_max   (C = sum_j T_j alpha_j c_j: the two terms of the derivative, T_i c_i and
//                                  -sum_{j>i} T_j alpha_j c_j / (1 - alpha_i), are each within [0, T_i c_max])
//   derived  = sum_i T_i alpha_i (c_max expm1(d w_i) + d colour_i)
// and widens the two fragile windows by the same uncertainty (alpha by d w, T' by the accumulated one). Depth order:
// two consecutive contributors may swap in the other record only if their z bit patterns are closer than the sum of
// their d z (equal bits with d z = 0 on both keep their index order on both sides); without slack the tie window is
// the flat 4 ulps of SURVEY.md 8(c).
constexpr int kSlack = 6;

// Oracle-R for one pixel over an ordered candidate list (Eq. 3, PAPER.md:L72;
// alpha PAPER.md:L79; depth / opacity targets PAPER.md:L87, L168; S9, S10, S12,
// S13, S16'). `budget` is the fragile-point allowance of DESIGN.md; `cond` is the
// fp32 conditioning allowance of the quadratic form.
PixelOut composite_pixel(const float* rec, const uint32_t* cand, size_t ncand, double px,
                         double py, const double bg[3], double c_max, bool tie_budget,
                         const double* slack = nullptr) {
  PixelOut o{};
  double T = 1.0, C[3] = {0, 0, 0}, D = 0.0;
  double relT = 0.0;   // accumulated relative uncertainty of T (end-to-end only)
  double prev_alpha = 0.0, prev_dz = 0.0;
  uint32_t prev_zbits = 0;
  bool have_prev = false;
  for (size_t k = 0; k < ncand; ++k) {
    const float* r = rec + (uint64_t)cand[k] * 12;
    ++o.visited;
    const double dx = (double)r[0] - px, dy = (double)r[1] - py;
    const double a = r[4], b = r[5], c = r[6];
    double w = -0.5 * (a * dx * dx + c * dy * dy) - b * dx * dy;
    if (w > 0.0) w = 0.0;  // S16': rounding guard, continuous (exact w <= 0)
    const double alpha = std::fmin(kAlphaMax, (double)r[3] * std::exp(w));
    double dw = 0.0, dcol = 0.0, dz = 0.0;
    if (slack) {
      const double* sl = slack + (uint64_t)cand[k] * kSlack;
      dw = std::fabs(a * dx + b * dy) * sl[0] + std::fabs(c * dy + b * dx) * sl[1] +
           (0.5 * dx * dx + 0.5 * dy * dy + std::fabs(dx * dy)) * sl[2] + sl[3];
      dcol = sl[4];
      dz = sl[5];
    }
    if (std::fabs(255.0 * alpha - 1.0) < 1e-4 + dw) o.budget += alpha * T * c_max;
    if (alpha < kAlphaMin) continue;
    const double Tn = T * (1.0 - alpha);
    const double dTn = relT + alpha * dw / (1.0 - alpha);   // relative uncertainty of T'
    if (std::fabs(Tn / kTStop - 1.0) < 1e-4 + dTn) o.budget += T * c_max;
    if (Tn < kTStop) break;  // S10: the Gaussian that would cross the stop is NOT composited
    const double wgt = alpha * T;
    o.derived += wgt * (c_max * std::expm1(dw) + dcol);
    relT = dTn;
    // fp32 evaluation of the quadratic form loses ~2^-22 of the sum of magnitudes
    o.cond += wgt * c_max * 2.384185791015625e-07 *
              (0.5 * (std::fabs(a) * dx * dx + std::fabs(c) * dy * dy) + std::fabs(b * dx * dy));
    if (tie_budget && have_prev) {
      const uint32_t zb = f32_bits(r[2]);
      const bool tie = slack ? (dz + prev_dz > 0.0 && (double)(zb - prev_zbits) <= dz + prev_dz) : (zb - prev_zbits <= 4u);
      // swapping two adjacent layers changes C by alpha_i alpha_j T_before (c_j - c_i), T_before = the
      // transmittance in front of BOTH = T / (1 - alpha_i)
      if (tie) o.budget += prev_alpha * alpha * (T / (1.0 - prev_alpha)) * c_max;
    }
    C[0] += (double)r[8] * wgt;
    C[1] += (double)r[9] * wgt;
    C[2] += (double)r[10] * wgt;
    D += (double)r[2] * wgt;
    T = Tn;
    ++o.contributed;
    prev_alpha = alpha;
    prev_zbits = f32_bits(r[2]);
    prev_dz = dz;
    have_prev = true;
  }
  o.alpha = 1.0 - T;
  for (int ch = 0; ch < 3; ++ch) o.rgb[ch] = C[ch] + T * bg[ch];
  o.depth = o.alpha > 0.0 ? D / o.alpha : 0.0;
  return o;
}

}  // namespace

extern "C" {

int oracle_record_stride() { return S_STRIDE; }

// Oracle-P: per-Gaussian state at time t and its projection (steps P1..P12 of
// DESIGN.md; Eq. 6, Eq. 7, Sigma PAPER.md:L79,
// Eq. 2, H(t) PAPER.md:L101/L120).
//   wide  [n][32] double : every intermediate (enum Slot)
//   rec32 [n][12] float  : (mx,my,z,op | a,b,c,hx | r,g,b,hy), zeros if culled
//
// oracle_preprocess_state adds the two variants of SURVEY.md 8(f-1):
//   dts != 0: the temporal-smoothing state H^(t2 = t) = { mu~(t1) + vbar dts, q, s, o~(t1), c } with
//             t1 = t - dts (Eq. 12) and vbar = v exp(-rho/2), rho = beta / l (Eq. 10; L112);
//   staticness filter: only points with rho_min <= rho <= rho_max are kept ("we remove the PVG points
//             whose rho < 1 to preserve the static part"; threshold on rho, L118).
//             beta = +INF is rho = +INF (3DGS, L114); l = +INF with finite beta is rho = 0.
void oracle_preprocess_state(uint64_t n, const float* mu, const float* quat, const float* scale,
                             const float* opacity, const float* sh, const float* tau,
                             const float* beta, const float* vel, double cycle, int sh_degree,
                             const Cam* cam, double t, double dts, double rho_min, double rho_max,
                             double* wide, float* rec32);

void oracle_preprocess(uint64_t n, const float* mu, const float* quat, const float* scale,
                       const float* opacity, const float* sh, const float* tau,
                       const float* beta, const float* vel, double cycle, int sh_degree,
                       const Cam* cam, double t, double* wide, float* rec32) {
  oracle_preprocess_state(n, mu, quat, scale, opacity, sh, tau, beta, vel, cycle, sh_degree, cam, t, 0.0, 0.0,
                          std::numeric_limits<double>::infinity(), wide, rec32);
}

void oracle_preprocess_state(uint64_t n, const float* mu, const float* quat, const float* scale,
                             const float* opacity, const float* sh, const float* tau,
                             const float* beta, const float* vel, double cycle, int sh_degree,
                             const Cam* cam, double t, double dts, double rho_min, double rho_max,
                             double* wide, float* rec32) {
  const double* R = cam->w2c;
  const int TX = (cam->width + kTile - 1) / kTile, TY = (cam->height + kTile - 1) / kTile;
  const double znear = cam->znear > 0.0 ? cam->znear : 0.2;  // S5
  // camera centre c_cam = -R^T T (P11)
  const double Tv[3] = {R[3], R[7], R[11]};
  double ccam[3];
  for (int j = 0; j < 3; ++j) ccam[j] = -(R[0 + j] * Tv[0] + R[4 + j] * Tv[1] + R[8 + j] * Tv[2]);
  const double limx = 1.3 * cam->width / (2.0 * cam->fx);   // S15
  const double limy = 1.3 * cam->height / (2.0 * cam->fy);
  const int ncoef = (sh_degree + 1) * (sh_degree + 1);

#pragma omp parallel for schedule(static)
  for (int64_t ii = 0; ii < (int64_t)n; ++ii) {
    const uint64_t i = (uint64_t)ii;
    double* w = wide + i * S_STRIDE;
    float* r32 = rec32 + i * 12;
    for (int k = 0; k < S_STRIDE; ++k) w[k] = 0.0;
    for (int k = 0; k < 12; ++k) r32[k] = 0.0f;
    w[S_RECT + 2] = w[S_RECT + 3] = -1.0;

    // P1: Eq. 6; l = +INF is the linear model
    // (Eq. 12: the state is evaluated at t1 = t - dts; dts = 0 is H(t) itself)
    const double dt = (t - dts) - (double)tau[i];
    const double m = std::isinf(cycle) ? dt : (cycle / (2.0 * kPi)) * std::sin(2.0 * kPi * dt / cycle);
    double mt[3];
    for (int j = 0; j < 3; ++j) mt[j] = (double)mu[i * 3 + j] + m * (double)vel[i * 3 + j];
    // P2: Eq. 7; beta = +INF => o~ = o
    const double be = beta[i];
    // staticness rho = beta / l
    const double rho = std::isinf(be) ? std::numeric_limits<double>::infinity() : (std::isinf(cycle) ? 0.0 : be / cycle);
    if (dts != 0.0) {
      // Eq. 10: vbar = v exp(-rho / 2); Eq. 12 (L162): flow translation vbar * dts
      const double e = std::exp(-0.5 * rho);
      for (int j = 0; j < 3; ++j) mt[j] += (double)vel[i * 3 + j] * e * dts;
    }
    if (!(rho >= rho_min) || rho > rho_max) { w[S_CULL] = 6; continue; }
    const double ot = std::isinf(be) ? (double)opacity[i]
                                     : (double)opacity[i] * std::exp(-0.5 * dt * dt / (be * be));
    for (int j = 0; j < 3; ++j) w[S_MU + j] = mt[j];
    w[S_OP] = ot;
    if (!finite3(mt) || !std::isfinite(ot)) { w[S_CULL] = 5; continue; }
    // P3: opacity cull (alpha <= o~ < 1/255 everywhere)
    if (!(ot >= kAlphaMin)) { w[S_CULL] = 1; continue; }
    // P4: camera space, near cull ("depth in camera space")
    double p[3];
    for (int j = 0; j < 3; ++j) p[j] = R[4 * j] * mt[0] + R[4 * j + 1] * mt[1] + R[4 * j + 2] * mt[2] + R[4 * j + 3];
    for (int j = 0; j < 3; ++j) w[S_PCAM + j] = p[j];
    if (!finite3(p)) { w[S_CULL] = 5; continue; }
    if (!(p[2] > znear)) { w[S_CULL] = 2; continue; }
    // P5: Sigma = R(q) diag(s^2) R(q)^T, q normalised
    double q[4] = {quat[i * 4], quat[i * 4 + 1], quat[i * 4 + 2], quat[i * 4 + 3]};
    const double qn = std::sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    for (int j = 0; j < 4; ++j) q[j] /= qn;
    const double qw = q[0], qx = q[1], qy = q[2], qz = q[3];
    const double Rq[9] = {1 - 2 * (qy * qy + qz * qz), 2 * (qx * qy - qw * qz), 2 * (qx * qz + qw * qy),
                          2 * (qx * qy + qw * qz), 1 - 2 * (qx * qx + qz * qz), 2 * (qy * qz - qw * qx),
                          2 * (qx * qz - qw * qy), 2 * (qy * qz + qw * qx), 1 - 2 * (qx * qx + qy * qy)};
    const double s2[3] = {(double)scale[i * 3] * scale[i * 3], (double)scale[i * 3 + 1] * scale[i * 3 + 1],
                          (double)scale[i * 3 + 2] * scale[i * 3 + 2]};
    double Sg[9];
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) {
        double acc = 0.0;
        for (int k = 0; k < 3; ++k) acc += Rq[a * 3 + k] * s2[k] * Rq[b * 3 + k];
        Sg[a * 3 + b] = acc;
      }
    w[S_SIG + 0] = Sg[0]; w[S_SIG + 1] = Sg[1]; w[S_SIG + 2] = Sg[2];
    w[S_SIG + 3] = Sg[4]; w[S_SIG + 4] = Sg[5]; w[S_SIG + 5] = Sg[8];
    // P6: Sigma' = J W Sigma W^T J^T (Eq. 2) + 0.3 I (S6); J guard S15
    const double z = p[2];
    const double xb = z * std::fmin(limx, std::fmax(-limx, p[0] / z));
    const double yb = z * std::fmin(limy, std::fmax(-limy, p[1] / z));
    const double J[6] = {cam->fx / z, 0.0, -cam->fx * xb / (z * z), 0.0, cam->fy / z, -cam->fy * yb / (z * z)};
    double Tm[6];  // T = J * W (2x3), W = rotation part of E
    for (int a = 0; a < 2; ++a)
      for (int b = 0; b < 3; ++b)
        Tm[a * 3 + b] = J[a * 3] * R[b] + J[a * 3 + 1] * R[4 + b] + J[a * 3 + 2] * R[8 + b];
    double TS[6];
    for (int a = 0; a < 2; ++a)
      for (int b = 0; b < 3; ++b)
        TS[a * 3 + b] = Tm[a * 3] * Sg[b] + Tm[a * 3 + 1] * Sg[3 + b] + Tm[a * 3 + 2] * Sg[6 + b];
    const double cxx = TS[0] * Tm[0] + TS[1] * Tm[1] + TS[2] * Tm[2] + kDilate;
    const double cxy = TS[0] * Tm[3] + TS[1] * Tm[4] + TS[2] * Tm[5];
    const double cyy = TS[3] * Tm[3] + TS[4] * Tm[4] + TS[5] * Tm[5] + kDilate;
    w[S_COV] = cxx; w[S_COV + 1] = cxy; w[S_COV + 2] = cyy;
    // P7: conic = Sigma'^-1
    const double det = cxx * cyy - cxy * cxy;
    if (!(det > 0.0) || !std::isfinite(det)) { w[S_CULL] = 3; continue; }
    const double ca = cyy / det, cb = -cxy / det, cc = cxx / det;
    w[S_CONIC] = ca; w[S_CONIC + 1] = cb; w[S_CONIC + 2] = cc;
    // P8: pinhole mean
    const double mx = cam->fx * p[0] / z + cam->cx, my = cam->fy * p[1] / z + cam->cy;
    w[S_MEAN] = mx; w[S_MEAN + 1] = my;
    // P9: exact-cutoff axis-aligned extents (S7)
    const double kk = 2.0 * std::log(255.0 * ot);
    const double hx = std::sqrt(kk * cxx), hy = std::sqrt(kk * cyy);
    w[S_EXT] = hx; w[S_EXT + 1] = hy;
    if (!std::isfinite(mx) || !std::isfinite(my) || !std::isfinite(hx) || !std::isfinite(hy)) { w[S_CULL] = 5; continue; }
    // P10: tile rectangle
    int tx0 = (int)std::floor(std::fmin(std::fmax((mx - hx) / kTile, -1.0), (double)TX));
    int tx1 = (int)std::floor(std::fmin(std::fmax((mx + hx) / kTile, -1.0), (double)TX));
    int ty0 = (int)std::floor(std::fmin(std::fmax((my - hy) / kTile, -1.0), (double)TY));
    int ty1 = (int)std::floor(std::fmin(std::fmax((my + hy) / kTile, -1.0), (double)TY));
    tx0 = std::max(tx0, 0); ty0 = std::max(ty0, 0);
    tx1 = std::min(tx1, TX - 1); ty1 = std::min(ty1, TY - 1);
    if (tx0 > tx1 || ty0 > ty1) { w[S_CULL] = 4; continue; }
    w[S_RECT] = tx0; w[S_RECT + 1] = ty0; w[S_RECT + 2] = tx1; w[S_RECT + 3] = ty1;
    w[S_COUNT] = (double)(tx1 - tx0 + 1) * (double)(ty1 - ty0 + 1);
    // P11: SH colour, view direction from mu~(t) (S3)
    double d[3] = {mt[0] - ccam[0], mt[1] - ccam[1], mt[2] - ccam[2]};
    const double dn = std::sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    for (int j = 0; j < 3; ++j) d[j] /= dn;
    double Y[16];
    sh_basis(d, Y);
    double rgb[3];
    for (int ch = 0; ch < 3; ++ch) {
      double acc = 0.0;
      for (int k = 0; k < ncoef; ++k) acc += Y[k] * (double)sh[(i * 16 + k) * 3 + ch];
      rgb[ch] = std::fmax(0.0, 0.5 + acc);
      w[S_RGB + ch] = rgb[ch];
    }
    if (!finite3(rgb)) { w[S_CULL] = 5; w[S_COUNT] = 0; continue; }
    // P12 + record rounded to fp32
    r32[0] = (float)mx; r32[1] = (float)my; r32[2] = (float)z; r32[3] = (float)ot;
    r32[4] = (float)ca; r32[5] = (float)cb; r32[6] = (float)cc; r32[7] = (float)hx;
    r32[8] = (float)rgb[0]; r32[9] = (float)rgb[1]; r32[10] = (float)rgb[2]; r32[11] = (float)hy;
  }
}

void oracle_sh_basis(const double* d, double* Y) { sh_basis(d, Y); }

// Integer chain, step 1: per-Gaussian tile rectangle + count from an fp32 record.
// Returns M = sum of counts.
// exact != 0: only the tiles of the rectangle that pass the P13 test are counted.
uint64_t oracle_tile_counts_ex(uint64_t n, const float* rec, int width, int height, int exact, int32_t* rects,
                               uint32_t* counts) {
  const int TX = (width + kTile - 1) / kTile, TY = (height + kTile - 1) / kTile;
  uint64_t M = 0;
  for (uint64_t i = 0; i < n; ++i) {
    int rc[4];
    uint32_t c = rect_of(rec + i * 12, TX, TY, rc);
    if (c && exact) {
      const ExactTile e = exact_tile_params(rec + i * 12);
      c = 0;
      for (int ty = rc[1]; ty <= rc[3]; ++ty) {
        int lo, hi;
        exact_row_span(e, ty, rc[0], rc[2], lo, hi);
        if (hi >= lo) c += (uint32_t)(hi - lo + 1);
      }
    }
    if (rects) for (int k = 0; k < 4; ++k) rects[i * 4 + k] = rc[k];
    if (counts) counts[i] = c;
    M += c;
  }
  return M;
}
// Per-tile list lengths (how many Gaussians list the tile), directly from the per-Gaussian tile sets: the ranges of the
// sorted list are their exclusive scan in row-major tile order. For full-size checks, where the M instances cannot be
// sorted in seconds.
void oracle_tile_hist_ex(uint64_t n, const float* rec, int width, int height, int exact, uint64_t* per_tile) {
  const int TX = (width + kTile - 1) / kTile, TY = (height + kTile - 1) / kTile;
  for (int64_t t = 0; t < (int64_t)TX * TY; ++t) per_tile[t] = 0;
  for (uint64_t i = 0; i < n; ++i) {
    int rc[4];
    if (!rect_of(rec + i * 12, TX, TY, rc)) continue;
    const ExactTile e = exact_tile_params(rec + i * 12);
    for (int ty = rc[1]; ty <= rc[3]; ++ty) {
      int lo = rc[0], hi = rc[2];
      if (exact) exact_row_span(e, ty, rc[0], rc[2], lo, hi);
      for (int tx = lo; tx <= hi; ++tx) ++per_tile[(size_t)ty * TX + tx];
    }
  }
}
uint64_t oracle_tile_counts(uint64_t n, const float* rec, int width, int height, int32_t* rects, uint32_t* counts) {
  return oracle_tile_counts_ex(n, rec, width, height, 0, rects, counts);
}

// Integer chain, step 2: emission order -> exclusive offsets -> unsorted
// (key,value) list -> stable sort by key -> per-tile ranges (S11).
//   order_mode 0: Gaussians visited in index order
//   order_mode 1: Gaussians visited in (fp32 z bits, index) order
// key = (ty*TX+tx) << 32 | bits(z); value = Gaussian index; tiles of one
// Gaussian are emitted row-major (ty outer, tx inner).
// offsets[n]: exclusive offset of Gaussian i's first instance (0-count rows get
// the running offset at their position in the visiting order).
void oracle_keys_ex(uint64_t n, const float* rec, int width, int height, int order_mode, int exact,
                    uint64_t* offsets, uint64_t* keys_unsorted, uint32_t* vals_unsorted,
                    uint64_t* keys_sorted, uint32_t* vals_sorted, uint32_t* ranges) {
  const int TX = (width + kTile - 1) / kTile, TY = (height + kTile - 1) / kTile;
  std::vector<uint32_t> visit;
  if (order_mode == 0) {
    visit.resize(n);
    for (uint64_t i = 0; i < n; ++i) visit[i] = (uint32_t)i;
  } else {
    visit = depth_order(n, rec);
    // culled rows follow, in index order (they emit nothing)
    for (uint64_t i = 0; i < n; ++i)
      if (!(rec[i * 12 + 3] > 0.0f)) visit.push_back((uint32_t)i);
  }
  uint64_t off = 0;
  for (uint64_t v = 0; v < n; ++v) {
    const uint32_t g = visit[v];
    int rc[4];
    const uint32_t c = rect_of(rec + (uint64_t)g * 12, TX, TY, rc);
    if (offsets) offsets[g] = off;
    const uint64_t zb = f32_bits(rec[(uint64_t)g * 12 + 2]);
    uint64_t o = off;
    if (c) {
      const ExactTile e = exact_tile_params(rec + (uint64_t)g * 12);
      for (int ty = rc[1]; ty <= rc[3]; ++ty) {
        int lo = rc[0], hi = rc[2];
        if (exact) exact_row_span(e, ty, rc[0], rc[2], lo, hi);
        for (int tx = lo; tx <= hi; ++tx) {
          keys_unsorted[o] = ((uint64_t)(ty * TX + tx) << 32) | zb;
          vals_unsorted[o] = g;
          ++o;
        }
      }
    }
    off = o;
  }
  const uint64_t M = off;
  std::vector<uint64_t> idx(M);
  for (uint64_t i = 0; i < M; ++i) idx[i] = i;
  std::stable_sort(idx.begin(), idx.end(),
                   [&](uint64_t a, uint64_t b) { return keys_unsorted[a] < keys_unsorted[b]; });
  for (uint64_t i = 0; i < M; ++i) {
    keys_sorted[i] = keys_unsorted[idx[i]];
    vals_sorted[i] = vals_unsorted[idx[i]];
  }
  const uint64_t ntiles = (uint64_t)TX * TY;
  for (uint64_t tl = 0; tl < ntiles; ++tl) {
    const uint64_t lo = std::lower_bound(keys_sorted, keys_sorted + M, tl << 32) - keys_sorted;
    const uint64_t hi = std::lower_bound(keys_sorted, keys_sorted + M, (tl + 1) << 32) - keys_sorted;
    ranges[tl * 2] = (uint32_t)lo;
    ranges[tl * 2 + 1] = (uint32_t)hi;
  }
}

void oracle_keys(uint64_t n, const float* rec, int width, int height, int order_mode,
                 uint64_t* offsets, uint64_t* keys_unsorted, uint32_t* vals_unsorted,
                 uint64_t* keys_sorted, uint32_t* vals_sorted, uint32_t* ranges) {
  oracle_keys_ex(n, rec, width, height, order_mode, 0, offsets, keys_unsorted, vals_unsorted, keys_sorted, vals_sorted, ranges);
}

// One tile's sorted instance list computed directly (no global sort): every
// non-culled Gaussian whose rectangle contains the tile, ascending by
// (fp32 z bits, index). Used for sampled full-size parity. Returns the length;
// writes at most `cap` entries.
uint64_t oracle_tile_list_ex(uint64_t n, const float* rec, int width, int height, uint32_t tile, int exact,
                             uint64_t cap, uint64_t* keys, uint32_t* vals) {
  const int TX = (width + kTile - 1) / kTile, TY = (height + kTile - 1) / kTile;
  const int tx = (int)(tile % TX), ty = (int)(tile / TX);
  std::vector<uint32_t> cand;
  for (uint64_t i = 0; i < n; ++i) {
    int rc[4];
    if (rect_of(rec + i * 12, TX, TY, rc) && tx >= rc[0] && tx <= rc[2] && ty >= rc[1] && ty <= rc[3]) {
      if (exact) {
        int lo, hi;
        exact_row_span(exact_tile_params(rec + i * 12), ty, rc[0], rc[2], lo, hi);
        if (tx < lo || tx > hi) continue;
      }
      cand.push_back((uint32_t)i);
    }
  }
  std::stable_sort(cand.begin(), cand.end(), [&](uint32_t a, uint32_t b) {
    return f32_bits(rec[(uint64_t)a * 12 + 2]) < f32_bits(rec[(uint64_t)b * 12 + 2]);
  });
  for (uint64_t k = 0; k < cand.size() && k < cap; ++k) {
    keys[k] = ((uint64_t)tile << 32) | f32_bits(rec[(uint64_t)cand[k] * 12 + 2]);
    vals[k] = cand[k];
  }
  return cand.size();
}
uint64_t oracle_tile_list(uint64_t n, const float* rec, int width, int height, uint32_t tile,
                          uint64_t cap, uint64_t* keys, uint32_t* vals) {
  return oracle_tile_list_ex(n, rec, width, height, tile, 0, cap, keys, vals);
}

// Oracle-R. mode 0 = brute force (every pixel visits every non-culled Gaussian in
// depth order); mode 1 = binned (a pixel visits only the Gaussians whose P10
// rectangle contains its tile, same order). tiles == nullptr renders the whole
// image, else only the listed tile ids (other pixels stay 0).
// Outputs are double: rgb [3][H][W], depth/alpha/budget/cond/derived [H][W].
// stats[0] = visited pairs, stats[1] = contributing pairs.
void oracle_render(uint64_t n, const float* rec, int width, int height, const double* bg, int mode,
                   const uint32_t* tiles, uint64_t ntiles_sel, int tie_budget, double* rgb,
                   double* depth, double* alpha, double* budget, double* cond, uint64_t* stats,
                   const double* slack /* [n][6] or nullptr: see kSlack */, double* derived /* [H][W] or nullptr */) {
  const int TX = (width + kTile - 1) / kTile, TY = (height + kTile - 1) / kTile;
  const uint64_t HW = (uint64_t)width * height;
  std::fill(rgb, rgb + 3 * HW, 0.0);
  std::fill(depth, depth + HW, 0.0);
  std::fill(alpha, alpha + HW, 0.0);
  if (budget) std::fill(budget, budget + HW, 0.0);
  if (cond) std::fill(cond, cond + HW, 0.0);
  if (derived) std::fill(derived, derived + HW, 0.0);
  const std::vector<uint32_t> order = depth_order(n, rec);
  double c_max = 0.0;
  for (uint32_t g : order)
    for (int ch = 0; ch < 3; ++ch) c_max = std::fmax(c_max, (double)rec[(uint64_t)g * 12 + 8 + ch]);
  for (int ch = 0; ch < 3; ++ch) c_max = std::fmax(c_max, bg[ch]);

  std::vector<uint32_t> sel;
  if (tiles) sel.assign(tiles, tiles + ntiles_sel);
  else { sel.resize((size_t)TX * TY); for (size_t k = 0; k < sel.size(); ++k) sel[k] = (uint32_t)k; }

  // binned: per selected tile, the Gaussians whose rectangle contains it, in depth order
  std::vector<std::vector<uint32_t>> lists;
  if (mode >= 1) {   // 1: binned by the P10 rectangle; 2: binned by the tiles that pass the P13 test (f-4)
    lists.resize(sel.size());
    std::vector<int32_t> slot((size_t)TX * TY, -1);
    for (size_t s = 0; s < sel.size(); ++s) slot[sel[s]] = (int32_t)s;
    for (uint32_t g : order) {
      int rc[4];
      if (!rect_of(rec + (uint64_t)g * 12, TX, TY, rc)) continue;
      const ExactTile e = exact_tile_params(rec + (uint64_t)g * 12);
      for (int ty = rc[1]; ty <= rc[3]; ++ty) {
        int lo = rc[0], hi = rc[2];
        if (mode == 2) exact_row_span(e, ty, rc[0], rc[2], lo, hi);
        for (int tx = lo; tx <= hi; ++tx) {
          const int32_t s = slot[(size_t)ty * TX + tx];
          if (s >= 0) lists[s].push_back(g);
        }
      }
    }
  }
  uint64_t visited = 0, contributed = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : visited, contributed)
  for (int64_t s = 0; s < (int64_t)sel.size(); ++s) {
    const int tx = (int)(sel[s] % TX), ty = (int)(sel[s] / TX);
    const uint32_t* cand = order.data();
    size_t ncand = order.size();
    if (mode >= 1) {
      cand = lists[s].data();
      ncand = lists[s].size();
    }
    for (int py = ty * kTile; py < std::min((ty + 1) * kTile, height); ++py)
      for (int px = tx * kTile; px < std::min((tx + 1) * kTile, width); ++px) {
        // S14: pixel centres at half-integers
        const PixelOut o = composite_pixel(rec, cand, ncand, px + 0.5, py + 0.5, bg, c_max, tie_budget != 0, slack);
        const uint64_t pi = (uint64_t)py * width + px;
        for (int ch = 0; ch < 3; ++ch) rgb[ch * HW + pi] = o.rgb[ch];
        depth[pi] = o.depth;
        alpha[pi] = o.alpha;
        if (budget) budget[pi] = o.budget;
        if (cond) cond[pi] = o.cond;
        if (derived) derived[pi] = o.derived;
        visited += o.visited;
        contributed += o.contributed;
      }
  }
  if (stats) { stats[0] = visited; stats[1] = contributed; }
}

// f-3: sky. "we utilize a high-resolution learnable environment cube map f_sky(d) = c_sky as
// the background. The final color is C_f = C + (1 - O) f_sky(d)"; "the sky color depends
// solely on the viewing direction". The paper fixes neither the cube-map layout nor the filter; readings
// (S20-S22):
//   d     = R^T ((px + 0.5 - cx) / fx, (py + 0.5 - cy) / fy, 1): the pixel-centre ray in world coordinates;
//   face  = 2 a + (d_a < 0), a = the axis of largest |d_a| (ties: lowest axis); the other two axes in cyclic
//           order (x -> y,z; y -> z,x; z -> x,y) give u = d_b / |d_a|, v = d_c / |d_a| in [-1, 1];
//   texel (i, j) of a face of resolution R has its centre at u = (2 i + 1) / R - 1, v = (2 j + 1) / R - 1;
//           cube[face][j][i][ch]; bilinear between the four nearest centres, clamped to the face.
// sky_sample is the definition written out; oracle_sky_composite applies C_f to an Oracle-R image rendered
// with bg = 0 (then rgb = C and alpha = O).
void oracle_sky_sample(const float* cube, int res, const double d[3], double out[3]) {
  int a = 0;
  if (std::fabs(d[1]) > std::fabs(d[a])) a = 1;
  if (std::fabs(d[2]) > std::fabs(d[a])) a = 2;
  const int b = (a + 1) % 3, c = (a + 2) % 3;
  const double m = std::fabs(d[a]);
  const int face = 2 * a + (d[a] < 0.0 ? 1 : 0);
  const double u = d[b] / m, v = d[c] / m;
  // continuous texel coordinates: centre of texel i is at s = i
  double sx = (u + 1.0) * 0.5 * res - 0.5, sy = (v + 1.0) * 0.5 * res - 0.5;
  sx = std::fmin(std::fmax(sx, 0.0), (double)(res - 1));
  sy = std::fmin(std::fmax(sy, 0.0), (double)(res - 1));
  const int i0 = (int)std::floor(sx), j0 = (int)std::floor(sy);
  const int i1 = std::min(i0 + 1, res - 1), j1 = std::min(j0 + 1, res - 1);
  const double fx = sx - i0, fy = sy - j0;
  const float* F = cube + (size_t)face * res * res * 3;
  for (int ch = 0; ch < 3; ++ch) {
    const double c00 = F[((size_t)j0 * res + i0) * 3 + ch], c10 = F[((size_t)j0 * res + i1) * 3 + ch];
    const double c01 = F[((size_t)j1 * res + i0) * 3 + ch], c11 = F[((size_t)j1 * res + i1) * 3 + ch];
    out[ch] = (1.0 - fy) * ((1.0 - fx) * c00 + fx * c10) + fy * ((1.0 - fx) * c01 + fx * c11);
  }
}

// rgb [3][H][W] (= C, rendered with bg = 0) and alpha [H][W] (= O) -> rgb += (1 - O) f_sky(d), in place
void oracle_sky_composite(const Cam* cam, const float* cube, int res, double* rgb, const double* alpha) {
  const double* R = cam->w2c;
  const uint64_t HW = (uint64_t)cam->width * cam->height;
  for (int py = 0; py < cam->height; ++py)
    for (int px = 0; px < cam->width; ++px) {
      const double dc[3] = {(px + 0.5 - cam->cx) / cam->fx, (py + 0.5 - cam->cy) / cam->fy, 1.0};
      double d[3];
      for (int j = 0; j < 3; ++j) d[j] = R[0 + j] * dc[0] + R[4 + j] * dc[1] + R[8 + j] * dc[2];   // R^T d_cam
      double sky[3];
      oracle_sky_sample(cube, res, d, sky);
      const uint64_t pi = (uint64_t)py * cam->width + px;
      for (int ch = 0; ch < 3; ++ch) rgb[ch * HW + pi] += (1.0 - alpha[pi]) * sky[ch];
    }
}

// f-2: the per-point quantities of the paper's dynamic element analysis, rendered by "replacing
// the color c in Eq. (3)": "we first transform vbar ... from the world coordinate system to the
// camera coordinate system" (L298), vbar = v exp(-rho / 2) (Eq. 10), rho = beta / l (L112); "we need to
// clamp each point's rho to the range of [0,2] and render" (L298). out[i] = (vbar_cam.x, .y, .z, clamp(rho, 0, 2));
// a velocity is a direction: only the rotation part of E applies. Rendering them is Oracle-R on a record whose
// colour slot holds these values, with bg = 0 (the sums of Eq. 3, no normalisation).
void oracle_dynamics(uint64_t n, const float* beta, const float* vel, double cycle, const Cam* cam, double* out) {
  const double* R = cam->w2c;
  for (uint64_t i = 0; i < n; ++i) {
    const double be = beta[i];
    const double rho = std::isinf(be) ? std::numeric_limits<double>::infinity() : (std::isinf(cycle) ? 0.0 : be / cycle);
    const double e = std::exp(-0.5 * rho);
    const double vb[3] = {vel[i * 3] * e, vel[i * 3 + 1] * e, vel[i * 3 + 2] * e};
    for (int j = 0; j < 3; ++j) out[i * 4 + j] = R[4 * j] * vb[0] + R[4 * j + 1] * vb[1] + R[4 * j + 2] * vb[2];
    out[i * 4 + 3] = std::fmin(std::fmax(rho, 0.0), 2.0);
  }
}

int oracle_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void oracle_set_threads(int nt) {
#ifdef _OPENMP
  if (nt > 0) omp_set_num_threads(nt);
#else
  (void)nt;
#endif
}

}  // extern "C"

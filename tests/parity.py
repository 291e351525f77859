"""Parity protocol between the CUDA path (through the C ABI binding) and the CPU oracle.

Three comparisons per frame:
  (P) GPU per-Gaussian record vs Oracle-P (double), with fragile points listed;
  (I) bit-exact integer chain: the integer oracle fed the GPU's own fp32 record vs the GPU's
      counts, offsets, unsorted keys, sorted keys/values and tile ranges;
  (R) GPU images vs Oracle-R fed the GPU record (isolates stages 2-5), and vs Oracle-R fed
      Oracle-P's record (end to end, nothing shared), both with the fragile budget.
"""
from __future__ import annotations

import numpy as np

import oracle
from oracle import SLOTS

TOL_RGB = 2e-4      # north_star: max-abs per colour channel
TOL_DEPTH_REL = 1e-3
EPS = 2.0 ** -23
EPS_D = 2.0 ** -52
CONIC_C = 64.0      # conic error model C eps amp (derivation at conic_tolerance): C = 24 covered the fp32 kernel of
                    # round 1 (EMPIRICAL: measured 11.7 at config 3, 10.2 at config 1); the record's conic is now
                    # computed in double, the same model applies with eps = 2^-52 and a wider C = 64
OP_REL = 3e-6       # o~: fp32 on the exact t - tau; the exponent of a survivor is > -5.5, three roundings of it ~1e-6
RGB_ABS = 5e-6      # SH colour, fp32 (measured 3e-7)
Z_REL = 1e-11       # two double evaluations of z = R (mu + m v) + T: a few 2^-53 of terms up to |mu| / z ~ 5000 times z


def f32_args(scene, t, dt=0.0, rho_min=0.0, rho_max=float("inf")):
    """The boundary's scalar arguments are C floats (include/pvg.h: pvg_scene_desc.cycle, pvg_render's t, pvg_state):
    the oracle must be evaluated at exactly the values the library receives, not at the Python doubles they were
    rounded from (t = k/49 is not an fp32 number; 0.2 is not either). Returns (cycle, t, dt, rho_min, rho_max)."""
    r = lambda x: float(np.float32(x))  # noqa: E731
    return r(scene.cycle), r(t), r(dt), r(rho_min), r(rho_max)


def oracle_preprocess(scene, cam, t, dt=0.0, rho_min=0.0, rho_max=float("inf")):
    """Oracle-P on the scene at the fp32 scalar arguments the C ABI receives."""
    cyc, t, dt, rho_min, rho_max = f32_args(scene, t, dt, rho_min, rho_max)
    return oracle.preprocess(scene.mu, scene.quat, scene.scale, scene.opacity, scene.sh, scene.tau, scene.beta,
                             scene.vel, cyc, scene.sh_degree, cam, t, dt, rho_min, rho_max)


def _rounding_fragile(x64: np.ndarray, rel: float = 1e-9, absolute=0.0) -> np.ndarray:
    """True where the double x lies within rel * (|x| + 1) + absolute of a midpoint between two adjacent fp32 numbers:
    there a second double computation of the same quantity (that far away) may round to the other neighbour."""
    f = x64.astype(np.float32).astype(np.float64)
    ulp = np.spacing(np.abs(x64).astype(np.float32)).astype(np.float64)
    return 0.5 * ulp - np.abs(x64 - f) < rel * (np.abs(x64) + 1.0) + absolute


def conic_tolerance(wide, scene, cam, sel):
    """How far two DOUBLE computations of the conic may differ, relative to sqrt(a c) kappa (kappa = Sigma'xx Sigma'yy /
    det): the covariance U U^T (U = J W R(q) diag(s)) carries an absolute error of C eps |T_row|^2 s_max^2 per entry,
    |T_row|^2 <= (f/z)^2 (1 + tx^2 + ty^2); relative to the smaller diagonal entry that is C eps amp, with amp >= 1
    large for needles seen end-on."""
    w = wide[sel]
    cov = w[:, SLOTS["cov"]]
    zc = w[:, 6]
    f = max(float(cam.fx), float(cam.fy))
    smax = scene.scale[sel].astype(np.float64).max(1)
    limx, limy = 1.3 * int(cam.width) / (2.0 * float(cam.fx)), 1.3 * int(cam.height) / (2.0 * float(cam.fy))
    txc, tyc = np.clip(w[:, 4] / zc, -limx, limx), np.clip(w[:, 5] / zc, -limy, limy)
    amp = (f / zc) ** 2 * (1.0 + txc ** 2 + tyc ** 2) * smax ** 2 / np.minimum(cov[:, 0], cov[:, 2])
    return CONIC_C * EPS_D * np.maximum(amp, 1.0)


def _conic_fragile(wide, scene, cam, sel):
    """[len(sel), 3] bool: conic entries that sit on an fp32 rounding midpoint up to the double-precision uncertainty."""
    w = wide[sel]
    cov, conic = w[:, SLOTS["cov"]], w[:, SLOTS["conic"]]
    kappa = cov[:, 0] * cov[:, 2] / (cov[:, 0] * cov[:, 2] - cov[:, 1] ** 2)
    tol_abs = conic_tolerance(wide, scene, cam, sel) * np.sqrt(conic[:, 0] * conic[:, 2]) * kappa
    return np.stack([_rounding_fragile(conic[:, j], rel=1e-12, absolute=tol_abs) for j in range(3)], 1)


def e2e_slack(wide: np.ndarray, scene, cam) -> np.ndarray:
    """Per-Gaussian distance allowed between the CUDA path's fp32 record and Oracle-P's, for the end-to-end image
    comparison (oracle.render(slack=...)); every column is the bound check_record asserts on the GPU record, computed
    from the oracle's own double values:
      d mx, d my, d conic : these run in double on both sides, so the two fp32 values are roundings of the same real
                   number up to ~1e-13: equal, unless that number sits on a rounding midpoint (then 1 ulp);
      d ln o~    : OP_REL;   d colour : RGB_ABS;
      d z        : 1 ulp where z sits on a rounding midpoint (two Gaussians whose depth bits are that close may then
                   be visited in the other order), else 0."""
    n = wide.shape[0]
    sl = np.zeros((n, 6), dtype=np.float64)
    v = wide[:, SLOTS["cull"]] == 0
    idx = np.nonzero(v)[0]
    w = wide[idx]
    ulp = lambda x: np.spacing(np.abs(x).astype(np.float32)).astype(np.float64)  # noqa: E731
    for col, slot in ((0, 19), (1, 20)):
        sl[idx, col] = np.where(_rounding_fragile(w[:, slot]), ulp(w[:, slot]), 0.0)
    conic = w[:, SLOTS["conic"]]
    sl[idx, 2] = np.where(_conic_fragile(wide, scene, cam, idx), ulp(conic), 0.0).max(1)
    sl[idx, 3] = OP_REL
    sl[idx, 4] = RGB_ABS
    sl[idx, 5] = np.where(_rounding_fragile(w[:, 6], rel=Z_REL), 1.0, 0.0)
    return sl


def check_record(gpu_rec: np.ndarray, wide: np.ndarray, cam, scene):
    """(P). Returns stats; raises AssertionError on a non-fragile mismatch."""
    n = gpu_rec.shape[0]
    width, height = int(cam.width), int(cam.height)
    znear = float(cam.znear) if cam.znear > 0 else 0.2
    o_valid = wide[:, SLOTS["cull"]] == 0
    g_valid = gpu_rec[:, 3] > 0
    # cull-fragile: o~*255, z/znear within 1e-5 of 1, or the tile rectangle within 1e-3 px of flipping empty
    op, z = wide[:, SLOTS["op"]], wide[:, 6]
    mx, my, hx, hy = wide[:, 19], wide[:, 20], wide[:, 21], wide[:, 22]
    TX, TY = (width + 15) // 16, (height + 15) // 16
    with np.errstate(invalid="ignore"):
        edge = np.stack([(mx - hx) / 16, (mx + hx) / 16, (my - hy) / 16, (my + hy) / 16], 1)
        rect_frag = np.any(np.abs(edge - np.round(edge)) < 1e-4, axis=1)
        cull_frag = (np.abs(op * 255 - 1) < 1e-5) | (np.abs(z / znear - 1) < 1e-5) | rect_frag
    mism = o_valid != g_valid
    bad = mism & ~cull_frag
    assert not bad.any(), f"cull mismatch on non-fragile Gaussians: {np.nonzero(bad)[0][:10]}"
    both = o_valid & g_valid
    g = gpu_rec[both].astype(np.float64)
    w = wide[both]
    stats = dict(n=n, survivors_gpu=int(g_valid.sum()), survivors_oracle=int(o_valid.sum()),
                 cull_mismatch_fragile=int(mism.sum()))
    if not both.any():
        return stats
    cov = w[:, SLOTS["cov"]]
    kappa = cov[:, 0] * cov[:, 2] / (cov[:, 0] * cov[:, 2] - cov[:, 1] ** 2)   # conditioning of the conic
    err = {}
    err["mean_px"] = np.abs(g[:, 0:2] - w[:, SLOTS["mean"]]).max(1)
    err["z_rel"] = np.abs(g[:, 2] - w[:, 6]) / w[:, 6]
    err["op_rel"] = np.abs(g[:, 3] - w[:, 3]) / w[:, 3]
    conic = w[:, SLOTS["conic"]]
    cn = np.sqrt(conic[:, 0] * conic[:, 2])
    err["conic_rel"] = np.abs(g[:, 4:7] - conic).max(1) / cn / kappa
    err["ext_rel"] = np.maximum(np.abs(g[:, 7] - w[:, 21]) / w[:, 21], np.abs(g[:, 11] - w[:, 22]) / w[:, 22])
    err["rgb_abs"] = np.abs(g[:, 8:11] - w[:, SLOTS["rgb"]]).max(1)
    for k, v in err.items():
        stats["max_" + k] = float(v.max())
    # mean and depth: the chain mu~(t) -> p_cam -> (mx, my) runs in double in the kernel as in the oracle, so the
    # fp32 record values are roundings of the same real number up to ~1e-13: BIT-EQUAL to the oracle's rounded record,
    # except where that number sits within 1e-9 relative of a rounding midpoint (then the neighbouring fp32 value)
    ulp = lambda x: np.spacing(np.abs(x).astype(np.float32)).astype(np.float64)  # noqa: E731
    for name, gcol, wcol in (("mx", 0, 19), ("my", 1, 20), ("z", 2, 6)):
        exact = g[:, gcol] == w[:, wcol].astype(np.float32).astype(np.float64)
        frag = _rounding_fragile(w[:, wcol], rel=Z_REL if name == "z" else 1e-9)
        stats[f"{name}_not_bit_equal"] = int((~exact).sum())
        assert np.all(exact | frag), (name, "not the correctly rounded value", int((~exact & ~frag).sum()))
        assert np.all(np.abs(g[:, gcol] - w[:, wcol]) <= 1.0001 * ulp(w[:, wcol])), (name, "more than 1 ulp off")
    assert err["op_rel"].max() <= OP_REL, ("opacity", stats["max_op_rel"])
    # conic: computed in double in the kernel (record passes) as in the oracle: bit-equal to the oracle's rounded
    # conic except on rounding midpoints, where the double-precision uncertainty is conic_tolerance's model
    cfrag = _conic_fragile(wide, scene, cam, both)
    cexact = g[:, 4:7] == conic.astype(np.float32).astype(np.float64)
    stats["conic_not_bit_equal"] = int((~cexact).sum())
    assert np.all(cexact | cfrag), ("conic not the correctly rounded value", int((~cexact & ~cfrag).sum()),
                                    stats["max_conic_rel"])
    assert np.all(np.abs(g[:, 4:7] - conic) <= 1.0001 * ulp(conic)), "conic more than 1 ulp off"
    # h = sqrt(2 ln(255 o~) Sigma'): near the opacity cutoff the logarithm is ~0 and carries an
    # absolute fp32 error of ~1e-6, i.e. a relative error 1e-6 / k in k and half that in h
    kk = 2.0 * np.log(255.0 * w[:, 3])
    ext_tol = 2e-5 + 2e-6 / np.maximum(kk, 1e-12)
    assert np.all(err["ext_rel"] <= ext_tol), ("extent", float((err["ext_rel"] / ext_tol).max()))
    assert err["rgb_abs"].max() <= RGB_ABS, ("rgb", stats["max_rgb_abs"])
    return stats


def check_integer_chain(dbg: dict, width: int, height: int, presort: bool, exact: bool = False):
    """(I): bit-exact. dbg = Scene.debug() of a render with KEEP_UNSORTED=1. exact: the exact tile lists (P13,
    PVG_OPT_EXACT_TILES): counts, offsets, sorted list and ranges of the refined tile sets; no unsorted list."""
    rec = dbg["record"]
    rects, counts, M = oracle.tile_counts(rec, width, height, exact)
    assert dbg["M"] == M, (dbg["M"], M)
    assert np.array_equal(dbg["counts"], counts), "per-Gaussian tile counts"
    k = oracle.keys(rec, width, height, 1 if presort else 0, exact=exact)
    n = rec.shape[0]
    if presort:
        visit = dbg["visit_order"]
        # survivors come first in (z bits, index) order; the culled tail is in index order
        rect_counts = oracle.tile_counts(rec, width, height)[1] if exact else counts   # survival is decided by the rectangle
        surv = np.nonzero(rect_counts)[0]
        exp = surv[np.lexsort((surv, rec[surv, 2].view(np.uint32)))]
        culled = np.nonzero(rect_counts == 0)[0]
        assert np.array_equal(visit, np.concatenate([exp, culled]).astype(np.uint32)), "depth visit order"
        off_by_g = np.empty(n, dtype=np.uint64)
        off_by_g[visit] = dbg["offsets"].astype(np.uint64)
    else:
        assert dbg["visit_order"] is None
        off_by_g = dbg["offsets"].astype(np.uint64)
    nz = counts > 0
    assert np.array_equal(off_by_g[nz], k["offsets"][nz]), "exclusive offsets"
    if dbg.get("keys_unsorted") is not None and M:
        assert np.array_equal(dbg["keys_unsorted"], k["keys_unsorted"]), "unsorted keys"
        assert np.array_equal(dbg["vals_unsorted"], k["vals_unsorted"]), "unsorted values"
    assert np.array_equal(dbg["keys_sorted"], k["keys_sorted"]), "sorted keys"
    assert np.array_equal(dbg["vals_sorted"], k["vals_sorted"]), "sorted values"
    assert np.array_equal(dbg["ranges"], k["ranges"]), "tile ranges"
    return dict(M=M, max_count=int(counts.max()), mean_list=float(M / max(1, k["ranges"].shape[0])))


def fragile_cap(rec: np.ndarray, ora: dict, pixels: int, end_to_end: bool = False) -> float:
    """Derived cap on the share of pixels with a non-zero fragile budget ("must be << 1 %" -- true of
    configs 0-3; the share grows with the number of list entries a pixel visits, so it is derived, not fixed).
    A visited (pixel, entry) pair is flagged when alpha is within 1e-4 relative of 1/255, i.e. when the pixel lies in
    the ring q0 (1 -+ 2e-4 / q0) of the Gaussian's Mahalanobis distance q = d^T Sigma'^-1 d, q0 = 2 ln(255 o~): an area of
    4e-4 pi sqrt(det Sigma') out of the 4 hx hy of the rectangle that made the pair a candidate. With p_ring the
    rectangle-area-weighted mean of that ratio over the record, the expected number of flags is visited * p_ring, and
    the share of flagged pixels is at most that over the pixel count (union bound). The pairs a pixel visits before
    it saturates are the FRONT of the scene, whose ring-to-rectangle ratio is not the record's average (measured flags
    are 0.8-2.2 times the expectation over configs 0-4), so the cap is three times the expectation plus three Poisson
    deviations plus 0.1 % for the T-stop window; end to end, where the windows are widened by the record uncertainty
    and reachable depth swaps are flagged too, another 0.5 % of the pixels."""
    live = rec[:, 3] > 0
    r = rec[live].astype(np.float64)
    det_conic = np.maximum(r[:, 4] * r[:, 6] - r[:, 5] ** 2, 1e-300)
    ring = 4e-4 * np.pi / np.sqrt(det_conic)            # sqrt(det Sigma') = 1 / sqrt(det conic)
    rect = 4.0 * r[:, 7] * r[:, 11]
    p_ring = float(ring.sum() / max(rect.sum(), 1e-300))
    expect = ora["visited"] * p_ring
    count = 3.0 * expect + 3.0 * np.sqrt(3.0 * expect) + 2.0 + (6e-3 if end_to_end else 1e-3) * pixels
    return float(min(1.0, count / max(pixels, 1)))


def check_images(gpu, ora, z_max: float, tol_rgb: float = TOL_RGB, with_cond: bool = True, label: str = "",
                 max_fragile_frac: float = 0.01):
    """(R): per pixel |rgb_gpu - rgb_oracle| <= tol + budget (+ fp32 conditioning allowance),
    depth within 1e-3 relative + budget * z_max / alpha. gpu = (rgb, depth, alpha) float32 arrays."""
    rgb, depth, alpha = (np.asarray(x, dtype=np.float64) for x in gpu)
    allow = ora["budget"] + (ora["cond"] if with_cond else 0.0) + ora.get("derived", 0.0)
    # budget and cond are weights (alpha T) times the colour scale c_max; alpha and depth flip by the bare weight
    allow_w = allow / ora["c_max"] if ora.get("c_max", 0.0) > 0 else allow
    e_rgb = np.abs(rgb - ora["rgb"]).max(0)
    e_alpha = np.abs(alpha - ora["alpha"])
    a = np.maximum(ora["alpha"], 1.0 / 255.0)
    e_depth = np.abs(depth - ora["depth"])
    depth_tol = TOL_DEPTH_REL * ora["depth"] + (np.maximum(allow, allow_w) + tol_rgb) * z_max / a
    clean = ora["budget"] == 0
    stats = dict(label=label,
                 max_rgb_err=float(e_rgb.max()), max_rgb_err_clean=float(e_rgb[clean].max()) if clean.any() else 0.0,
                 max_alpha_err=float(e_alpha.max()),
                 max_depth_rel=float((e_depth / np.maximum(ora["depth"], 1e-9))[ora["alpha"] > 0].max()) if (ora["alpha"] > 0).any() else 0.0,
                 fragile_pixels=int((~clean).sum()), pixels=int(clean.size),
                 max_cond=float(ora["cond"].max()),
                 max_derived=float(np.max(ora.get("derived", 0.0))))
    bad_rgb = e_rgb > tol_rgb + allow
    bad_alpha = e_alpha > tol_rgb + np.maximum(allow, allow_w)
    bad_depth = e_depth > depth_tol
    stats["bad_rgb"], stats["bad_alpha"], stats["bad_depth"] = int(bad_rgb.sum()), int(bad_alpha.sum()), int(bad_depth.sum())
    assert not bad_rgb.any(), ("rgb", stats)
    assert not bad_alpha.any(), ("alpha", stats)
    assert not bad_depth.any(), ("depth", stats)
    # the share of pixels with a non-zero budget grows with the number of candidates per pixel (each one is a
    # chance to land within 1e-4 of a threshold): 0.4-0.6 % at configs 0-3, a few % at the stress config
    assert stats["fragile_pixels"] <= max_fragile_frac * stats["pixels"], ("too many fragile pixels", stats)
    return stats

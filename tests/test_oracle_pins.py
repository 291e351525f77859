"""Pins for the CPU oracle (oracle/pvg_oracle.cpp) against what the paper and the
mathematics fix: closed forms, invariants, library routines (scipy rotations,
scipy spherical harmonics, numpy stable sort / matrix inverse), Monte-Carlo and
brute force. None of these retypes the oracle's own formula. CPU only.

Citations: PAPER.md:L<line>; T1..T8 = SURVEY.md section 4; P/S/R = DESIGN.md readings.
"""
import math

import numpy as np
import pytest
from scipy.spatial.transform import Rotation
from scipy.special import sph_harm_y

import oracle
from oracle import SLOTS
from helpers import cam_simple, one_scene, record_row
from workloads import make_config, pinhole_camera

L = 0.2


def P(scene, cam, t):
    return oracle.preprocess_scene(scene, cam, t)


# ----------------------------------------------------------------------------- Eq. 6
class TestEq6:
    """mu~(t) = mu + l/(2 pi) sin(2 pi (t - tau)/l) v."""
    mu = np.array([0.5, -0.25, 6.0])
    v = np.array([1.5, -0.75, 0.5])
    tau = 0.25
    cam = cam_simple()

    def mut(self, t, cycle=L):
        sc = one_scene(mu=self.mu, vel=self.v, tau=self.tau, cycle=cycle)
        return P(sc, self.cam, t)[0][0, SLOTS["mu"]]

    def test_peak_at_tau(self):                      # T1
        assert np.array_equal(self.mut(self.tau), self.mu)

    def test_instant_velocity(self):                 # T2, PAPER.md:L110  v = d mu~/dt at tau
        h = 1e-5
        slope = (self.mut(self.tau + h) - self.mut(self.tau - h)) / (2 * h)
        assert np.allclose(slope, self.v, rtol=1e-6, atol=1e-8)

    def test_amplitude_quarter_cycle(self):          # sin = 1 at t - tau = l/4
        assert np.allclose(self.mut(self.tau + L / 4) - self.mu, L / (2 * math.pi) * self.v, rtol=1e-13)

    def test_twelfth_cycle(self):                    # sin(pi/6) = 1/2 pins the 2 pi inside the sine
        assert np.allclose(self.mut(self.tau + L / 12) - self.mu, L / (4 * math.pi) * self.v, rtol=1e-12)

    def test_bounded_by_v(self):                     # PAPER.md:L112 "bounded nature of mu~(t) by v"
        for t in np.linspace(-1, 2, 37):
            assert np.linalg.norm(self.mut(t) - self.mu) <= L / (2 * math.pi) * np.linalg.norm(self.v) * (1 + 1e-12)

    def test_periodic(self):                         # north_star: mu(t + l) = mu(t)
        for t in (0.03, 0.41, 0.77):
            assert np.allclose(self.mut(t + L), self.mut(t), atol=1e-13)

    def test_cycle_mean_is_mu(self):                 # T3, PAPER.md:L112  E[mu~] = mu over a multiple of l
        ts = 0.1 + (np.arange(64) + 0.5) / 64 * (2 * L)
        m = np.mean([self.mut(t) for t in ts], axis=0)
        assert np.allclose(m, self.mu, atol=1e-13)

    def test_linear_limit(self):                     # T5, PAPER.md:L336/L377  l -> inf is mu + v (t - tau)
        for dt in (-0.4, 0.1, 0.7):
            lin = self.mut(self.tau + dt, cycle=np.inf)
            assert np.allclose(lin, self.mu + dt * self.v, rtol=1e-14)
            big = self.mut(self.tau + dt, cycle=1e4)
            bound = np.linalg.norm(self.v) * abs(dt) ** 3 * (2 * math.pi / 1e4) ** 2 / 6
            assert np.linalg.norm(big - lin) <= bound * (1 + 1e-6) + 1e-15

    def test_static_when_v_zero(self):               # T4 half: v = 0 => mu~ = mu for every t
        sc = one_scene(mu=self.mu, vel=(0, 0, 0), tau=0.3)
        for t in (0.0, 0.5, 0.9):
            assert np.array_equal(P(sc, self.cam, t)[0][0, SLOTS["mu"]], self.mu)


# ----------------------------------------------------------------------------- Eq. 7
class TestEq7:
    """o~(t) = o exp(-(t - tau)^2 / (2 beta^2))."""
    cam = cam_simple()
    o, tau, beta = 0.75, 0.5, 0.125

    def ot(self, t, beta=None):
        sc = one_scene(opacity=self.o, tau=self.tau, beta=self.beta if beta is None else beta)
        return P(sc, self.cam, t)[0][0, SLOTS["op"]]

    def test_peak(self):                             # T1
        assert self.ot(self.tau) == self.o

    def test_symmetric(self):                        # T6 / north_star
        for d in (0.01, 0.1, 0.2):
            assert self.ot(self.tau + d) == pytest.approx(self.ot(self.tau - d), rel=1e-14)

    def test_one_and_two_sigma(self):                # e^{-1/2}, e^{-2}: pins the 1/2 and the square
        assert self.ot(self.tau + self.beta) == pytest.approx(self.o * math.exp(-0.5), rel=1e-14)
        assert self.ot(self.tau - 2 * self.beta) == pytest.approx(self.o * math.exp(-2.0), rel=1e-14)

    def test_decay_rate_inverse_in_beta(self):
        assert self.ot(self.tau + 0.1, beta=0.05) < self.ot(self.tau + 0.1, beta=0.1) < self.o

    def test_beta_inf_is_static(self):               # T4, PAPER.md:L114  rho = +inf
        assert self.ot(0.0, beta=np.inf) == self.o and self.ot(0.93, beta=np.inf) == self.o


# ----------------------------------------------------------------------------- Sigma
class TestSigma:
    """Sigma = R(q) diag(s^2) R(q)^T."""
    cam = cam_simple()

    @staticmethod
    def full(w):
        xx, xy, xz, yy, yz, zz = w[SLOTS["sigma"]]
        return np.array([[xx, xy, xz], [xy, yy, yz], [xz, yz, zz]])

    def test_identity_quat(self):
        s = np.array([0.5, 0.25, 0.125])
        w, _ = P(one_scene(scale=s), self.cam, 0.0)
        assert np.allclose(self.full(w[0]), np.diag(s ** 2), atol=1e-16)

    def test_against_scipy_rotation(self):
        rng = np.random.default_rng(7)
        for _ in range(20):
            q = rng.normal(size=4)                   # un-normalised on purpose: the oracle normalises
            s = np.exp(rng.normal(size=3)).astype(np.float32)
            q32 = q.astype(np.float32)
            w, _ = P(one_scene(quat=q32, scale=s), self.cam, 0.0)
            qd = q32.astype(np.float64)
            R = Rotation.from_quat([qd[1], qd[2], qd[3], qd[0]]).as_matrix()   # scipy: (x,y,z,w)
            S = R @ np.diag(s.astype(np.float64) ** 2) @ R.T
            assert np.allclose(self.full(w[0]), S, rtol=1e-12, atol=1e-14)
            assert np.trace(self.full(w[0])) == pytest.approx(np.sum(s.astype(np.float64) ** 2), rel=1e-12)
            assert np.linalg.det(self.full(w[0])) == pytest.approx(np.prod(s.astype(np.float64) ** 2), rel=1e-9)

    def test_quarter_turn_about_z_swaps_xy(self):
        c = math.sqrt(0.5)
        w, _ = P(one_scene(quat=(c, 0, 0, c), scale=(0.5, 0.25, 0.125)), self.cam, 0.0)
        assert np.allclose(self.full(w[0]), np.diag([0.25 ** 2, 0.5 ** 2, 0.125 ** 2]), atol=1e-8)


# ----------------------------------------------------------------------------- EWA
def rotated_camera(width=200, height=120, f=150.0):
    cam = pinhole_camera(width, height, f)
    R = Rotation.from_euler("xyz", [0.2, -0.3, 0.1]).as_matrix()
    T = np.array([0.3, -0.2, 0.5])
    cam.world_to_cam = np.concatenate([R, T[:, None]], axis=1).astype(np.float32).reshape(12)
    return cam


def project(cam, pw):
    E = np.asarray(cam.world_to_cam, dtype=np.float64).reshape(3, 4)
    pc = pw @ E[:, :3].T + E[:, 3]
    return np.stack([cam.fx * pc[..., 0] / pc[..., 2] + cam.cx, cam.fy * pc[..., 1] / pc[..., 2] + cam.cy], -1), pc


class TestEWA:
    """Sigma' = J W Sigma W^T J^T (+0.3 I)   (Eq. 2)."""

    @staticmethod
    def cov2(w):
        xx, xy, yy = w[SLOTS["cov"]]
        return np.array([[xx, xy], [xy, yy]])

    def test_isotropic_on_axis_closed_form(self):
        cam = cam_simple(64, 48, 50.0)
        s, z = 0.25, 5.0
        w, _ = P(one_scene(mu=(0, 0, z), scale=(s, s, s)), cam, 0.0)
        assert np.allclose(self.cov2(w[0]), ((50.0 * s / z) ** 2 + 0.3) * np.eye(2), rtol=1e-13)
        assert np.allclose(w[0, SLOTS["mean"]], [cam.cx, cam.cy])

    def test_mean_is_pinhole_projection(self):
        cam = rotated_camera()
        pw = np.array([0.4, -0.3, 7.0], dtype=np.float32)
        w, _ = P(one_scene(mu=pw), cam, 0.0)
        m, pc = project(cam, pw.astype(np.float64))
        assert np.allclose(w[0, SLOTS["mean"]], m, rtol=1e-13)
        assert np.allclose(w[0, SLOTS["pcam"]], pc, rtol=1e-13)

    def test_jacobian_by_finite_differences(self):
        # rank-1 Sigma = eps^2 e_k e_k^T  =>  Sigma' - 0.3 I = eps^2 (d pi / d e_k)(d pi / d e_k)^T
        cam = rotated_camera()
        pw = np.array([0.5, -0.25, 6.0], dtype=np.float32)
        eps, tiny, h = 0.125, 1e-9, 1e-6
        for k in range(3):
            s = np.full(3, tiny, dtype=np.float32)
            s[k] = eps
            w, _ = P(one_scene(mu=pw, scale=s), cam, 0.0)
            e = np.zeros(3)
            e[k] = 1.0
            g = (project(cam, pw + h * e)[0] - project(cam, pw - h * e)[0]) / (2 * h)
            assert np.allclose(self.cov2(w[0]) - 0.3 * np.eye(2), eps ** 2 * np.outer(g, g), rtol=1e-6, atol=1e-9)

    def test_monte_carlo_projected_covariance(self):
        cam = rotated_camera()
        pw = np.array([0.3, 0.2, 8.0], dtype=np.float32)
        q = np.array([0.9, 0.1, -0.3, 0.2], dtype=np.float32)
        s = np.array([0.04, 0.02, 0.01], dtype=np.float32)
        w, _ = P(one_scene(mu=pw, quat=q, scale=s), cam, 0.0)
        rng = np.random.default_rng(11)
        qd = q.astype(np.float64) / np.linalg.norm(q.astype(np.float64))
        R = Rotation.from_quat([qd[1], qd[2], qd[3], qd[0]]).as_matrix()
        pts = pw.astype(np.float64) + (rng.normal(size=(1_000_000, 3)) * s.astype(np.float64)) @ R.T
        uv, _ = project(cam, pts)
        emp = np.cov(uv.T)
        ref = self.cov2(w[0]) - 0.3 * np.eye(2)
        assert np.allclose(emp, ref, rtol=0, atol=0.01 * np.sqrt(ref[0, 0] * ref[1, 1]))

    def test_jacobian_guard_uses_clamped_ray(self):  # S15
        cam = cam_simple(64, 48, 50.0)
        z, s = 4.0, (0.2, 0.1, 0.3)
        lim = 1.3 * 64 / (2 * 50.0)
        far, _ = P(one_scene(mu=(5.0 * lim * z, 0, z), scale=s), cam, 0.0)
        edge, _ = P(one_scene(mu=(lim * z, 0, z), scale=s), cam, 0.0)
        assert np.allclose(far[0, SLOTS["cov"]], edge[0, SLOTS["cov"]], rtol=1e-6)

    def test_conic_is_inverse(self):
        cam = rotated_camera()
        w, _ = P(one_scene(mu=(0.2, 0.1, 4.0), quat=(0.7, 0.2, 0.5, -0.1), scale=(0.3, 0.05, 0.1)), cam, 0.0)
        a, b, c = w[0, SLOTS["conic"]]
        assert np.allclose(np.array([[a, b], [b, c]]), np.linalg.inv(self.cov2(w[0])), rtol=1e-10)


# ----------------------------------------------------------------------------- extents / tiles
class TestExtents:
    def test_tangent_points_have_cutoff_alpha(self):  # S7: AABB of the alpha = 1/255 ellipse
        cam = rotated_camera()
        w, _ = P(one_scene(mu=(0.2, 0.1, 4.0), quat=(0.7, 0.2, 0.5, -0.1), scale=(0.3, 0.05, 0.1), opacity=0.6), cam, 0.0)
        cov = TestEWA.cov2(w[0])
        ci = np.linalg.inv(cov)
        hx, hy = w[0, SLOTS["ext"]]
        ot = w[0, SLOTS["op"]]
        for d in (cov[:, 0] * hx / cov[0, 0], cov[:, 1] * hy / cov[1, 1]):   # tangent points on x = hx, y = hy
            assert ot * math.exp(-0.5 * d @ ci @ d) == pytest.approx(1 / 255, rel=1e-12)
        assert abs(cov[0, 0] * hx / cov[0, 0] - hx) < 1e-12

    def test_no_pixel_outside_rect_reaches_cutoff(self):
        wl = make_config(0)
        cam = wl.cameras[0]
        w, rec = P(wl.scene, cam, 0.37)
        ys, xs = np.mgrid[0:cam.height, 0:cam.width]
        px, py = xs + 0.5, ys + 0.5
        valid = np.nonzero(w[:, SLOTS["cull"]] == 0)[0]
        for g in valid[:400]:
            cov = TestEWA.cov2(w[g])
            ci = np.linalg.inv(cov)
            dx, dy = w[g, 19] - px, w[g, 20] - py
            alpha = w[g, SLOTS["op"]] * np.exp(-0.5 * (ci[0, 0] * dx * dx + 2 * ci[0, 1] * dx * dy + ci[1, 1] * dy * dy))
            tx0, ty0, tx1, ty1 = w[g, SLOTS["rect"]].astype(int)
            inside = (xs // 16 >= tx0) & (xs // 16 <= tx1) & (ys // 16 >= ty0) & (ys // 16 <= ty1)
            assert not np.any((alpha >= (1 / 255) * (1 + 1e-9)) & ~inside)

    def test_rect_is_interval_tile_overlap(self):    # P10 == brute-force tile membership
        wl = make_config(0)
        cam = wl.cameras[0]
        w, rec = P(wl.scene, cam, 0.0)
        TX, TY = cam.width // 16, cam.height // 16
        rects, counts, M = oracle.tile_counts(rec, cam.width, cam.height)
        for g in range(wl.scene.n):
            if rec[g, 3] <= 0:
                assert counts[g] == 0
                continue
            mx, my, hx, hy = (np.float64(rec[g, 0]), np.float64(rec[g, 1]), np.float64(rec[g, 7]), np.float64(rec[g, 11]))
            tiles_x = [t for t in range(TX) if mx - hx < 16 * t + 16 and mx + hx >= 16 * t]
            tiles_y = [t for t in range(TY) if my - hy < 16 * t + 16 and my + hy >= 16 * t]
            assert counts[g] == len(tiles_x) * len(tiles_y)
            if counts[g]:
                assert list(rects[g]) == [tiles_x[0], tiles_y[0], tiles_x[-1], tiles_y[-1]]
        assert M == counts.sum()

    def test_culls(self):
        cam = cam_simple()
        w, rec = P(one_scene(mu=[(0, 0, 5), (0, 0, 0.1), (0, 0, -3), (100, 0, 5), (0, 0, 5)],
                             opacity=[0.5, 0.5, 0.5, 0.5, 0.003]), cam, 0.0)
        assert list(w[:, SLOTS["cull"]].astype(int)) == [0, 2, 2, 4, 1]
        assert np.all(rec[1:] == 0) and rec[0, 3] == np.float32(0.5)

    def test_faded_point_is_culled(self):            # PVG-specific: o~(t) < 1/255 far from tau
        cam = cam_simple()
        sc = one_scene(opacity=0.9, tau=0.5, beta=0.02)
        assert P(sc, cam, 0.5)[0][0, SLOTS["cull"]] == 0
        assert P(sc, cam, 0.7)[0][0, SLOTS["cull"]] == 1


# ----------------------------------------------------------------------------- SH
def real_sh_scipy(d):
    """Real SH with the Condon-Shortley phase kept: k = l(l+1)+m,
    m>0: sqrt2 Re Y_l^m, m<0: sqrt2 Im Y_l^|m|, m=0: Y_l^0 (scipy.special.sph_harm_y)."""
    d = np.asarray(d, dtype=np.float64)
    theta, phi = math.acos(d[2]), math.atan2(d[1], d[0])
    out = np.zeros(16)
    for l in range(4):
        for m in range(-l, l + 1):
            y = sph_harm_y(l, abs(m), theta, phi)
            out[l * (l + 1) + m] = y.real if m == 0 else math.sqrt(2) * (y.real if m > 0 else y.imag)
    return out


class TestSH:
    def test_basis_matches_scipy(self):
        rng = np.random.default_rng(3)
        for _ in range(50):
            d = rng.normal(size=3)
            d /= np.linalg.norm(d)
            assert np.allclose(oracle.sh_basis(d), real_sh_scipy(d), atol=1e-13)

    def test_orthonormal_by_quadrature(self):
        zs, wz = np.polynomial.legendre.leggauss(8)
        nphi = 16
        G = np.zeros((16, 16))
        for z, wq in zip(zs, wz):
            for j in range(nphi):
                ph = 2 * math.pi * (j + 0.5) / nphi
                r = math.sqrt(1 - z * z)
                Y = oracle.sh_basis([r * math.cos(ph), r * math.sin(ph), z])
                G += wq * (2 * math.pi / nphi) * np.outer(Y, Y)
        assert np.allclose(G, np.eye(16), atol=1e-12)

    def test_pole(self):                             # only the m = 0 terms survive at d = +z
        Y = oracle.sh_basis([0, 0, 1.0])
        expect = np.zeros(16)
        expect[0] = math.sqrt(1 / (4 * math.pi))
        expect[2] = math.sqrt(3 / (4 * math.pi))
        expect[6] = 2 * math.sqrt(5 / (16 * math.pi))
        expect[12] = 2 * math.sqrt(7 / (16 * math.pi))
        assert np.allclose(Y, expect, atol=1e-15)

    def test_colour_dc_only_and_clamp(self):
        cam = cam_simple()
        sh = np.zeros((2, 16, 3), dtype=np.float32)
        sh[0, 0] = (1.0, -0.5, 0.25)
        sh[1, 0] = (-3.0, 0.0, 0.0)                  # 0.5 + Y0 * (-3) < 0 -> clamped to 0
        w, _ = P(one_scene(mu=[(0.3, 0.2, 5), (0, 0, 6)], sh=sh), cam, 0.0)
        y0 = 0.28209479177387814
        assert np.allclose(w[0, SLOTS["rgb"]], 0.5 + y0 * sh[0, 0].astype(np.float64), rtol=1e-14)
        assert w[1, 23] == 0.0 and w[1, 24] == 0.5

    def test_colour_view_direction_from_camera_centre(self):
        cam = rotated_camera()
        rng = np.random.default_rng(5)
        sh = (0.2 * rng.normal(size=(1, 16, 3))).astype(np.float32)
        pw = np.array([0.4, -0.3, 7.0], dtype=np.float32)
        v = np.array([2.0, 0.0, 1.0], dtype=np.float32)
        t, tau = 0.31, 0.25
        sc = one_scene(mu=pw, sh=sh, vel=v, tau=tau)
        w, _ = P(sc, cam, t)
        E4 = np.eye(4)
        E4[:3] = np.asarray(cam.world_to_cam, dtype=np.float64).reshape(3, 4)
        centre = np.linalg.inv(E4)[:3, 3]            # camera centre in world coordinates
        d = w[0, SLOTS["mu"]] - centre               # direction from mu~(t), not mu (S3)
        d /= np.linalg.norm(d)
        col = np.maximum(0.0, 0.5 + real_sh_scipy(d) @ sh[0].astype(np.float64))
        assert np.allclose(w[0, SLOTS["rgb"]], col, atol=1e-12)
        assert not np.allclose(w[0, SLOTS["mu"]], pw)

    def test_degree_truncation(self):
        cam = cam_simple()
        rng = np.random.default_rng(9)
        sh = (0.2 * rng.normal(size=(1, 16, 3))).astype(np.float32)
        for deg in range(4):
            trunc = sh.copy()
            trunc[:, (deg + 1) ** 2:] = 0
            a, _ = P(one_scene(mu=(0.5, 0.4, 5), sh=sh, sh_degree=deg), cam, 0.0)
            b, _ = P(one_scene(mu=(0.5, 0.4, 5), sh=trunc, sh_degree=3), cam, 0.0)
            assert np.array_equal(a[0, SLOTS["rgb"]], b[0, SLOTS["rgb"]])


# ----------------------------------------------------------------------------- blend (Oracle-R)
W, H = 32, 32


def flat(op, z, rgb=(1, 1, 1)):
    """A layer with alpha = op at every pixel (zero conic)."""
    return record_row(16.0, 16.0, z, op, 0.0, 0.0, 0.0, rgb)


def R(rows, mode="binned", bg=(0, 0, 0), w=W, h=H, **kw):
    return oracle.render(np.stack(rows), w, h, bg=bg, mode=mode, **kw)


class TestBlend:
    """C = sum T_i alpha_i c_i, T_i = prod_{j<i}(1 - alpha_j)   (Eq. 3)."""

    def test_R1_single_gaussian_image(self):
        cam = cam_simple(64, 48, 50.0)
        sh = np.zeros((1, 16, 3), dtype=np.float32)
        sh[0, 0] = (1.0, 0.2, -0.4)
        sc = one_scene(mu=(0.31, -0.17, 4.0), quat=(0.8, 0.1, 0.3, -0.5), scale=(0.4, 0.1, 0.2), opacity=0.9, sh=sh)
        w, rec = P(sc, cam, 0.0)
        out = oracle.render(rec, cam.width, cam.height, mode="brute")
        r = rec[0].astype(np.float64)
        ci = np.linalg.inv(np.linalg.inv(np.array([[r[4], r[5]], [r[5], r[6]]])))   # conic via two inversions
        ys, xs = np.mgrid[0:cam.height, 0:cam.width]
        d = np.stack([r[0] - (xs + 0.5), r[1] - (ys + 0.5)], -1)
        wq = -0.5 * np.einsum("...i,ij,...j->...", d, ci, d)
        alpha = np.minimum(0.99, r[3] * np.exp(wq))
        alpha[alpha < 1 / 255] = 0.0
        assert np.allclose(out["alpha"], alpha, atol=1e-12)
        for ch in range(3):
            assert np.allclose(out["rgb"][ch], alpha * r[8 + ch], atol=1e-12)
        assert np.allclose(out["depth"][alpha > 0], r[2], rtol=1e-12)
        assert np.all(out["depth"][alpha == 0] == 0)
        assert alpha.max() > 0.85 and (alpha == 0).any()
        # and the fp32 conic agrees with the double Sigma' it came from
        assert np.allclose(np.linalg.inv(ci), TestEWA.cov2(w[0]), rtol=1e-5)

    def test_R2_two_layers(self):
        a1, a2 = 0.25, 0.5
        c1, c2 = np.array([1.0, 0.0, 0.5]), np.array([0.0, 1.0, 0.25])
        out = R([flat(a1, 2.0, c1), flat(a2, 3.0, c2)])
        assert np.allclose(out["rgb"][:, 5, 7], a1 * c1 + (1 - a1) * a2 * c2, rtol=1e-14)
        assert out["alpha"][5, 7] == pytest.approx(1 - (1 - a1) * (1 - a2), rel=1e-14)
        assert out["depth"][5, 7] == pytest.approx((a1 * 2.0 + (1 - a1) * a2 * 3.0) / (a1 + (1 - a1) * a2), rel=1e-14)

    def test_depth_order_not_index_order(self):
        c1, c2 = (1.0, 0.0, 0.0), (0.0, 1.0, 0.0)
        near_first = R([flat(0.5, 2.0, c1), flat(0.5, 3.0, c2)])
        swapped = R([flat(0.5, 3.0, c2), flat(0.5, 2.0, c1)])
        assert np.array_equal(near_first["rgb"], swapped["rgb"])
        assert near_first["rgb"][0, 0, 0] == 0.5 and near_first["rgb"][1, 0, 0] == 0.25

    def test_depth_tie_lower_index_first(self):      # S11
        out = R([flat(0.5, 2.0, (1, 0, 0)), flat(0.5, 2.0, (0, 1, 0))])
        assert out["rgb"][0, 0, 0] == 0.5 and out["rgb"][1, 0, 0] == 0.25

    def test_R3_n_identical_layers(self):
        a, n = 0.125, 20
        out = R([flat(a, 1.0 + i, (0.5, 0.5, 0.5)) for i in range(n)])
        assert out["alpha"][3, 3] == pytest.approx(1 - (1 - a) ** n, rel=1e-13)
        assert out["rgb"][0, 3, 3] == pytest.approx(0.5 * (1 - (1 - a) ** n), rel=1e-13)

    def test_R4_stop_rule(self):                     # S10: the crossing Gaussian is not composited
        out = R([flat(0.8, 1.0 + i) for i in range(8)])
        a = float(np.float32(0.8))                   # 6th layer: T' = 6.4e-5 < 1e-4
        assert out["alpha"][0, 0] == pytest.approx(1 - (1 - a) ** 5, rel=1e-14)
        assert out["contributed"] == 5 * W * H

    def test_R5_alpha_clamp(self):                   # S9: 0.99
        out = R([flat(1.0, 1.0)])
        assert out["alpha"][0, 0] == pytest.approx(0.99, rel=1e-15)

    def test_R6_alpha_cutoff(self):                  # S9: 1/255
        assert R([flat(0.00391, 1.0)])["alpha"].max() == 0.0
        assert R([flat(0.00393, 1.0)])["alpha"].min() == pytest.approx(float(np.float32(0.00393)), rel=1e-15)

    def test_background(self):                       # S13 / PAPER.md:L168 with a constant f_sky
        out = R([flat(0.25, 1.0, (1.0, 1.0, 1.0))], bg=(0.2, 0.4, 0.8))
        assert np.allclose(out["rgb"][:, 1, 1], 0.25 + 0.75 * np.array([0.2, 0.4, 0.8]), rtol=1e-14)
        empty = oracle.render(np.zeros((1, 12), dtype=np.float32), W, H, bg=(0.2, 0.4, 0.8))
        assert np.allclose(empty["rgb"][:, 0, 0], [0.2, 0.4, 0.8]) and empty["alpha"].max() == 0

    @pytest.mark.parametrize("t", [0.0, 0.37, 0.5])
    def test_R7_brute_equals_binned_cfg0(self, t):
        wl = make_config(0)
        cam = wl.cameras[0]
        _, rec = P(wl.scene, cam, t)
        a = oracle.render(rec, cam.width, cam.height, mode="brute")
        b = oracle.render(rec, cam.width, cam.height, mode="binned")
        for k in ("rgb", "depth", "alpha"):
            assert np.array_equal(a[k], b[k])
        assert b["visited"] < a["visited"]

    def test_R7_brute_equals_binned_partial_tiles_and_subset(self):
        wl = make_config(1, n=3000)
        cam = pinhole_camera(150, 70, 120.0)         # 150 = 9*16+6, 70 = 4*16+6: ragged last tiles
        _, rec = P(wl.scene, cam, 0.5)
        a = oracle.render(rec, cam.width, cam.height, mode="brute")
        b = oracle.render(rec, cam.width, cam.height, mode="binned")
        assert np.array_equal(a["rgb"], b["rgb"]) and np.array_equal(a["alpha"], b["alpha"])
        sub = oracle.render(rec, cam.width, cam.height, mode="binned", tiles=[0, 9, 49])
        assert np.array_equal(sub["rgb"][:, 64:70, 144:150], a["rgb"][:, 64:70, 144:150])   # tile 49: last, ragged
        assert np.array_equal(sub["rgb"][:, 0:16, 0:16], a["rgb"][:, 0:16, 0:16])
        assert sub["alpha"][20, 40] == 0.0           # unselected tile left empty

    def test_R8_permutation_invariance(self):
        wl = make_config(0)
        cam = wl.cameras[0]
        _, rec = P(wl.scene, cam, 0.37)
        z = rec[rec[:, 3] > 0, 2]
        assert len(np.unique(z)) == len(z)           # no depth ties in this scene
        perm = np.random.default_rng(1).permutation(rec.shape[0])
        a = oracle.render(rec, cam.width, cam.height)
        b = oracle.render(rec[perm], cam.width, cam.height)
        assert np.array_equal(a["rgb"], b["rgb"]) and np.array_equal(a["depth"], b["depth"])

    def test_budget_flags_fragile_points_only(self):
        assert R([flat(0.5, 1.0)])["budget"].max() == 0.0
        assert R([flat(np.float32(1 / 255), 1.0)])["budget"].min() > 0.0      # alpha on the 1/255 edge
        # T' = 1e-4 exactly on the stop edge: 4 layers of 0.9 -> T = 1e-4 (within 1e-4 relative)
        assert R([flat(0.9, 1.0 + i) for i in range(4)])["budget"].min() > 0.0


# ----------------------------------------------------------------------------- whole render
class TestWholeRender:
    def setup_method(self):
        self.wl = make_config(0)
        self.cam = self.wl.cameras[0]

    def img(self, scene, t):
        _, rec = P(scene, self.cam, t)
        return oracle.render(rec, self.cam.width, self.cam.height)

    def test_t_equals_tau_is_static_3dgs(self):      # north_star / T1
        sc = self.wl.scene
        sc_tau = one_scene(mu=sc.mu, quat=sc.quat, scale=sc.scale, opacity=sc.opacity, sh=sc.sh,
                           tau=np.full(sc.n, 0.375, np.float32), beta=sc.beta, vel=sc.vel)
        static = one_scene(mu=sc.mu, quat=sc.quat, scale=sc.scale, opacity=sc.opacity, sh=sc.sh,
                           tau=np.zeros(sc.n, np.float32), beta=np.full(sc.n, np.inf, np.float32),
                           vel=np.zeros_like(sc.vel))
        a, b = self.img(sc_tau, 0.375), self.img(static, 0.9)
        assert np.array_equal(a["rgb"], b["rgb"]) and np.array_equal(a["depth"], b["depth"])

    def test_static_scene_independent_of_t(self):    # T4
        sc = self.wl.scene
        static = one_scene(mu=sc.mu, quat=sc.quat, scale=sc.scale, opacity=sc.opacity, sh=sc.sh, tau=sc.tau,
                           beta=np.full(sc.n, np.inf, np.float32), vel=np.zeros_like(sc.vel))
        a, b = self.img(static, 0.1), self.img(static, 0.83)
        assert np.array_equal(a["rgb"], b["rgb"])

    def test_periodic_when_opacity_constant(self):
        sc = self.wl.scene
        per = one_scene(mu=sc.mu, quat=sc.quat, scale=sc.scale, opacity=sc.opacity, sh=sc.sh, tau=sc.tau,
                        beta=np.full(sc.n, np.inf, np.float32), vel=sc.vel)
        a, b = self.img(per, 0.3), self.img(per, 0.3 + L)
        bud = a["budget"] + b["budget"]
        assert np.all(np.abs(a["rgb"] - b["rgb"]).max(0) <= 1e-9 + bud)
        assert not np.allclose(a["rgb"], self.img(per, 0.3 + L / 2)["rgb"], atol=1e-3)

    def test_opacity_symmetric_for_still_point(self):
        sc = one_scene(mu=(0.1, 0.2, 5), scale=(0.3, 0.2, 0.1), opacity=0.9, tau=0.5, beta=0.1,
                       sh=np.full((1, 16, 3), 0.1, np.float32))
        cam = cam_simple()
        a = oracle.render(P(sc, cam, 0.5 + 0.07)[1], cam.width, cam.height)
        b = oracle.render(P(sc, cam, 0.5 - 0.07)[1], cam.width, cam.height)
        assert np.allclose(a["rgb"], b["rgb"], atol=1e-7) and a["alpha"].max() > 0.3

    def test_linear_limit_render(self):              # T5: l -> inf equals rendering linearly moved points
        sc = self.wl.scene
        t = 0.5
        lin = one_scene(mu=sc.mu, quat=sc.quat, scale=sc.scale, opacity=sc.opacity, sh=sc.sh, tau=sc.tau,
                        beta=sc.beta, vel=sc.vel, cycle=np.inf)
        moved_mu = (sc.mu.astype(np.float64) + (t - sc.tau.astype(np.float64))[:, None] * sc.vel.astype(np.float64))
        wa, _ = P(lin, self.cam, t)
        assert np.allclose(wa[:, SLOTS["mu"]], moved_mu, rtol=1e-14)


# ----------------------------------------------------------------------------- integer chain
class TestIntegerChain:
    @pytest.mark.parametrize("order_mode", [0, 1])
    def test_chain_invariants_and_library_sort(self, order_mode):
        wl = make_config(0)
        cam = wl.cameras[0]
        _, rec = P(wl.scene, cam, 0.37)
        rects, counts, M = oracle.tile_counts(rec, cam.width, cam.height)
        k = oracle.keys(rec, cam.width, cam.height, order_mode)
        assert k["M"] == M == int(counts.sum())
        ku, vu, ks, vs, rg = k["keys_unsorted"], k["vals_unsorted"], k["keys_sorted"], k["vals_sorted"], k["ranges"]
        # library stable sort of the unsorted list
        idx = np.argsort(ku, kind="stable")
        assert np.array_equal(ks, ku[idx]) and np.array_equal(vs, vu[idx])
        assert np.all(np.diff(ks.astype(np.int64)) >= 0)
        # ranges tile the list
        assert rg[0, 0] == 0 and rg[-1, 1] == M and np.array_equal(rg[1:, 0], rg[:-1, 1])
        tile_of = (ks >> np.uint64(32)).astype(np.int64)
        for tl in range(rg.shape[0]):
            assert np.all(tile_of[rg[tl, 0]:rg[tl, 1]] == tl)
        # low word is the fp32 bit pattern of that Gaussian's depth
        assert np.array_equal((ks & np.uint64(0xFFFFFFFF)).astype(np.uint32), rec[vs, 2].view(np.uint32))
        # brute-force per-tile membership, ordered by (depth bits, index)
        TX = cam.width // 16
        zb = rec[:, 2].view(np.uint32)
        for tl in range(rg.shape[0]):
            tx, ty = tl % TX, tl // TX
            members = [g for g in range(rec.shape[0]) if counts[g] and rects[g, 0] <= tx <= rects[g, 2]
                       and rects[g, 1] <= ty <= rects[g, 3]]
            members.sort(key=lambda g: (int(zb[g]), g))
            assert list(vs[rg[tl, 0]:rg[tl, 1]]) == members
            kk, vv = oracle.tile_list(rec, cam.width, cam.height, tl)
            assert list(vv) == members and np.array_equal(kk, ks[rg[tl, 0]:rg[tl, 1]])

    def test_emission_order(self):
        wl = make_config(0)
        cam = wl.cameras[0]
        _, rec = P(wl.scene, cam, 0.0)
        rects, counts, M = oracle.tile_counts(rec, cam.width, cam.height)
        k0 = oracle.keys(rec, cam.width, cam.height, 0)
        assert np.array_equal(k0["offsets"], np.concatenate([[0], np.cumsum(counts.astype(np.uint64))[:-1]]))
        g = int(np.argmax(counts))
        o = int(k0["offsets"][g])
        TX = cam.width // 16
        tiles = [(ty * TX + tx) for ty in range(rects[g, 1], rects[g, 3] + 1) for tx in range(rects[g, 0], rects[g, 2] + 1)]
        assert list((k0["keys_unsorted"][o:o + counts[g]] >> np.uint64(32)).astype(int)) == tiles
        assert np.all(k0["vals_unsorted"][o:o + counts[g]] == g)
        # depth-ordered emission: values appear in (z bits, index) order of the survivors
        k1 = oracle.keys(rec, cam.width, cam.height, 1)
        firsts = k1["vals_unsorted"][np.concatenate([[True], np.diff(k1["vals_unsorted"].astype(np.int64)) != 0])]
        surv = np.nonzero(counts)[0]
        expect = surv[np.lexsort((surv, rec[surv, 2].view(np.uint32)))]
        assert np.array_equal(firsts, expect)

    def test_stable_ties(self):
        rows = [record_row(20.0, 20.0, 2.0, 0.5, 0.01, 0, 0.01, hx=10, hy=10) for _ in range(5)]
        k = oracle.keys(np.stack(rows), 64, 64, 0)
        for tl in range(k["ranges"].shape[0]):
            s, e = k["ranges"][tl]
            if e > s:
                assert list(k["vals_sorted"][s:e]) == [0, 1, 2, 3, 4]


# ----------------------------------------------------------------------------- f-1: Eq. 10 / Eq. 12, staticness filter
class TestTemporalSmoothingState:
    """H^(t2) = { mu~(t1) + vbar (t2 - t1), q, s, o~(t1), c }, vbar = v exp(-rho/2), rho = beta/l
    (Eq. 10, Eq. 12, rho L112); filter on rho (L118, L192)."""
    mu = np.array([0.5, -0.25, 6.0])
    v = np.array([1.5, -0.75, 0.5])
    tau = 0.25
    cam = cam_simple()

    def state(self, t, dt, beta, cycle=L, **kw):
        sc = one_scene(mu=self.mu, vel=self.v, tau=self.tau, beta=beta, cycle=cycle, opacity=0.8)
        w = oracle.preprocess_scene(sc, self.cam, t, dt, **kw)[0][0]
        return w[SLOTS["mu"]], w[SLOTS["op"]], int(w[SLOTS["cull"]])

    def test_dt_zero_is_the_plain_state(self):       # "assign a probability of eta to set dt as 0 (no estimation)", L166
        wl = make_config(0)
        a = oracle.preprocess_scene(wl.scene, wl.cameras[0], 0.37)
        b = oracle.preprocess_scene(wl.scene, wl.cameras[0], 0.37, 0.0)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])

    def test_opacity_is_taken_at_t1(self):           # Eq. 12: o~(t1), not o~(t2)
        for dt in (-0.03, 0.02):
            _, op_hat, _ = self.state(0.3, dt, beta=0.1)
            _, op_t1, _ = self.state(0.3 - dt, 0.0, beta=0.1)
            assert op_hat == op_t1

    def test_flow_translation(self):                 # Eq. 12 minus the plain state at t1 is vbar * dt; Eq. 10 for vbar
        for beta, dt in ((0.05, 0.02), (0.3, -0.015), (0.02, 0.01)):
            mu_hat, _, _ = self.state(0.31, dt, beta)
            mu_t1, _, _ = self.state(0.31 - dt, 0.0, beta)
            rho = float(np.float32(beta)) / L          # the model stores beta in fp32
            assert np.allclose(mu_hat - mu_t1, self.v * math.exp(-rho / 2) * dt, rtol=1e-11, atol=1e-16)

    def test_limits_of_the_average_velocity(self):   # T8: rho -> inf: vbar -> 0; rho -> 0: vbar -> v
        dt = 0.02
        mu_hat, _, _ = self.state(0.3, dt, beta=np.inf)
        mu_t1, _, _ = self.state(0.3 - dt, 0.0, beta=np.inf)
        assert np.array_equal(mu_hat, mu_t1)                                  # vbar = 0 exactly
        mu_hat, _, _ = self.state(0.3, dt, beta=1e-9)
        mu_t1, _, _ = self.state(0.3 - dt, 0.0, beta=1e-9)
        assert np.allclose(mu_hat - mu_t1, self.v * dt, rtol=1e-8)           # vbar = v

    def test_estimates_the_next_state_of_a_fast_point(self):
        """L160: 'dynamic objects often maintain a constant speed within a short time interval': for rho -> 0 and
        t1, t2 near tau the estimate equals the true state up to the curvature of the sine, |v| |D|^3 (2 pi / l)^2 / 6
        summed over the two ends."""
        beta, dt, t2 = 1e-6, 0.004, self.tau + 0.006
        mu_hat, _, _ = self.state(t2, dt, beta)
        mu_true, _, _ = self.state(t2, 0.0, beta)
        k = (2 * math.pi / L) ** 2 / 6
        bound = np.linalg.norm(self.v) * k * (abs(t2 - self.tau) ** 3 + abs(t2 - dt - self.tau) ** 3)
        assert 0 < np.linalg.norm(mu_hat - mu_true) <= bound * (1 + 1e-6)

    def test_linear_model_has_rho_zero(self):        # l = +inf: rho = beta / l = 0, vbar = v, and mu + v (t1 - tau) + v dt = mu + v (t2 - tau)
        mu_hat, _, _ = self.state(0.4, 0.05, beta=0.1, cycle=np.inf)
        assert np.allclose(mu_hat, self.mu + self.v * (0.4 - self.tau), rtol=1e-14)

    def test_staticness_filter(self):                # L192: "remove the PVG points whose rho < 1"
        assert self.state(0.25, 0.0, beta=0.19, rho_min=1.0)[2] == 6          # rho = 0.95: removed
        assert self.state(0.25, 0.0, beta=0.2, rho_min=1.0)[2] == 0           # rho = 1: kept (fp32 0.2 / 0.2)
        assert self.state(0.25, 0.0, beta=np.inf, rho_min=1.0)[2] == 0        # 3DGS point: rho = +inf (L114)
        assert self.state(0.25, 0.0, beta=0.5, rho_max=1.0)[2] == 6           # dynamic-only view drops static points
        assert self.state(0.25, 0.0, beta=0.1, rho_max=1.0)[2] == 0
        assert self.state(0.25, 0.0, beta=50.0, cycle=np.inf, rho_min=1e-3)[2] == 6   # l = inf: rho = 0

    def test_filter_partitions_the_scene(self):
        """rho < 1 and rho >= 1 partition the points: the two filtered records are disjoint and their union is the
        unfiltered record, row by row."""
        wl = make_config(0)
        cam = wl.cameras[0]
        full = oracle.preprocess_scene(wl.scene, cam, 0.37)[1]
        stat = oracle.preprocess_scene(wl.scene, cam, 0.37, 0.0, 1.0)[1]
        rho = wl.scene.beta.astype(np.float64) / wl.scene.cycle
        dyn = oracle.preprocess_scene(wl.scene, cam, 0.37, 0.0, 0.0, float(np.nextafter(1.0, 0.0)))[1]
        keep = rho >= 1.0
        assert np.array_equal(stat[keep], full[keep]) and not stat[~keep].any()
        assert np.array_equal(dyn[~keep], full[~keep]) and not dyn[keep].any()
        assert 0 < keep.sum() < len(keep)


# ----------------------------------------------------------------------------- f-3: sky cube map
class TestSky:
    """C_f = C + (1 - O) f_sky(d); cube-map layout and filter: DESIGN.md S20-S22."""

    @staticmethod
    def direction(face, u, v):
        a, sign = face // 2, (1.0 if face % 2 == 0 else -1.0)
        d = np.zeros(3)
        d[a], d[(a + 1) % 3], d[(a + 2) % 3] = sign, u, v
        return d

    def test_constant_map(self):
        cube = np.full((6, 8, 8, 3), 0.0, np.float32)
        cube[..., 0], cube[..., 1], cube[..., 2] = 0.25, 0.5, 0.75
        rng = np.random.default_rng(0)
        for d in rng.normal(size=(50, 3)):
            assert np.array_equal(oracle.sky_sample(cube, d), [0.25, 0.5, 0.75])

    def test_axis_directions_pick_their_face(self):
        cube = np.zeros((6, 4, 4, 3), np.float32)
        for f in range(6):
            cube[f] = f + 1
        for f in range(6):
            assert np.array_equal(oracle.sky_sample(cube, self.direction(f, 0.0, 0.0)), [f + 1] * 3)
            assert np.array_equal(oracle.sky_sample(cube, 7.5 * self.direction(f, 0.3, -0.8)), [f + 1] * 3)   # |d| irrelevant

    def test_texel_centres_return_the_texel(self):
        rng = np.random.default_rng(1)
        res = 16
        cube = rng.random((6, res, res, 3)).astype(np.float32)
        for _ in range(200):
            f, i, j = rng.integers(6), rng.integers(res), rng.integers(res)
            d = self.direction(f, (2 * i + 1) / res - 1, (2 * j + 1) / res - 1)
            assert np.allclose(oracle.sky_sample(cube, d), cube[f, j, i], rtol=0, atol=1e-12)

    def test_bilinear_reproduces_affine_faces(self):
        res = 32
        i, j = np.meshgrid(np.arange(res), np.arange(res), indexing="xy")
        cube = np.zeros((6, res, res, 3), np.float32)
        for f in range(6):
            cube[f, ..., 0], cube[f, ..., 1], cube[f, ..., 2] = i, j, 0.5 * i - 0.25 * j + f   # exact in fp32
        rng = np.random.default_rng(2)
        lim = 1 - 1 / res                                   # between the outermost texel centres
        for _ in range(200):
            f, u, v = rng.integers(6), rng.uniform(-lim, lim), rng.uniform(-lim, lim)
            si, sj = (u + 1) / 2 * res - 0.5, (v + 1) / 2 * res - 0.5
            got = oracle.sky_sample(cube, self.direction(f, u, v))
            assert np.allclose(got, [si, sj, 0.5 * si - 0.25 * sj + f], rtol=0, atol=1e-10)

    def test_clamped_at_the_face_edge(self):
        res = 8
        i, j = np.meshgrid(np.arange(res), np.arange(res), indexing="xy")
        cube = np.zeros((6, res, res, 3), np.float32)
        cube[0, ..., 0], cube[0, ..., 1] = i, j
        got = oracle.sky_sample(cube, self.direction(0, 0.999999, 0.0))      # beyond the last centre: edge value
        assert np.allclose(got[:2], [res - 1, (0 + 1) / 2 * res - 0.5], atol=1e-9)

    def test_composite_weights_by_one_minus_opacity(self):
        cam = cam_simple(64, 48, 50.0)
        rec = np.stack([record_row(32.3, 24.2, 3.0, 0.7, 0.02, 0.0, 0.02, rgb=(0.2, 0.4, 0.6))])
        base = oracle.render(rec, cam.width, cam.height, mode="brute")
        cube = np.zeros((6, 4, 4, 3), np.float32)
        cube[4] = (0.1, 0.3, 0.9)                          # +z face: identity pose looks down +z, FoV < 45 deg
        out = oracle.sky_composite(cam, cube, base["rgb"], base["alpha"])
        sky = np.array([0.1, 0.3, 0.9], np.float32).astype(np.float64)       # the map holds fp32 values
        expect = base["rgb"] + (1 - base["alpha"])[None] * sky[:, None, None]
        assert np.allclose(out, expect, rtol=0, atol=1e-15)
        # a constant map is a constant background: ties the sky to the pinned bg path (S13)
        const = np.zeros((6, 4, 4, 3), np.float32)
        const[...] = (0.5, 0.25, 0.125)
        with_bg = oracle.render(rec, cam.width, cam.height, bg=(0.5, 0.25, 0.125), mode="brute")
        assert np.allclose(oracle.sky_composite(cam, const, base["rgb"], base["alpha"]), with_bg["rgb"], rtol=0, atol=1e-15)

    def test_direction_is_in_world_coordinates(self):
        """Camera yawed by +90 deg (camera->world = R_y: camera +z points along world +x): an empty frame shows the +x face."""
        cube = np.zeros((6, 4, 4, 3), np.float32)
        for f in range(6):
            cube[f] = f + 1
        zero = np.zeros((3, 48, 64)), np.zeros((48, 64))
        for yaw, face in ((0.0, 4), (90.0, 0), (-90.0, 1), (180.0, 5)):
            cam = pinhole_camera(64, 48, 50.0, yaw_deg=yaw)
            out = oracle.sky_composite(cam, cube, *zero)
            assert np.all(out[:, 20:28, 28:36] == face + 1), (yaw, out[0, 24, 32])


# ----------------------------------------------------------------------------- f-2: velocity / staticness targets
class TestDynamicsTarget:
    """vbar = v exp(-rho/2) in camera axes and clamp(rho, 0, 2), rendered by replacing c in Eq. 3."""

    def test_limits_and_clamp(self):                 # T8 (L156) and the [0, 2] clamp (L298)
        cam = cam_simple()
        sc = one_scene(mu=[(0, 0, 5)] * 4, vel=[(1.0, -2.0, 0.5)] * 4, beta=[np.inf, 1e-9, 0.1, 0.7])
        f = oracle.dynamics(sc, cam)
        assert np.array_equal(f[0], [0, 0, 0, 2.0])                                   # rho = inf: vbar = 0, clamp at 2
        assert np.allclose(f[1], [1.0, -2.0, 0.5, 0.0], rtol=1e-8, atol=5e-9)         # rho -> 0: vbar = v
        assert np.allclose(f[2, :3], np.array([1.0, -2.0, 0.5]) * math.exp(-float(np.float32(0.1)) / L / 2), rtol=1e-13)
        assert f[2, 3] == float(np.float32(0.1)) / L and f[3, 3] == 2.0               # 0.5 inside, 3.5 clamped

    def test_velocity_rotates_but_does_not_translate(self):
        sc = one_scene(mu=(0, 0, 5), vel=(3.0, 0.0, 0.0), beta=1e-9)
        # camera yawed +90 deg looks along world +x: a world +x velocity points INTO that camera (+z), no x/y part
        f = oracle.dynamics(sc, pinhole_camera(64, 48, 50.0, yaw_deg=90.0))[0]
        assert np.allclose(f[:3], [0.0, 0.0, 3.0], atol=1e-6)
        cam = cam_simple()
        moved = cam_simple()
        moved.world_to_cam = cam.world_to_cam.copy()
        moved.world_to_cam[[3, 7, 11]] = (5.0, -2.0, 9.0)                             # translation only
        assert np.array_equal(oracle.dynamics(sc, cam), oracle.dynamics(sc, moved))

    def test_rendering_is_eq3_with_the_colour_replaced(self):
        """One Gaussian: the velocity image is alpha(x) * vbar_cam, the staticness image alpha(x) * clamp(rho)."""
        cam = cam_simple(64, 48, 50.0)
        sc = one_scene(mu=(0.1, 0.05, 3.0), scale=(0.2, 0.1, 0.1), opacity=0.9, vel=(-1.5, 0.25, 2.0), beta=0.06)
        _, rec = oracle.preprocess_scene(sc, cam, 0.0)
        f = oracle.dynamics(sc, cam)
        plain = oracle.render(rec, cam.width, cam.height, mode="brute")              # alpha image of the single Gaussian
        r = rec.copy()
        r[:, 8:11] = f[:, :3]
        vel_img = oracle.render(r, cam.width, cam.height, mode="brute")["rgb"]
        r[:, 8] = f[:, 3]
        rho_img = oracle.render(r, cam.width, cam.height, mode="brute")["rgb"][0]
        a = plain["alpha"]
        for ch in range(3):
            assert np.allclose(vel_img[ch], a * float(np.float32(f[0, ch])), rtol=1e-12, atol=1e-15)
        assert np.allclose(rho_img, a * float(np.float32(f[0, 3])), rtol=1e-12, atol=1e-15) and a.max() > 0.8


# ----------------------------------------------------------------------------- end-to-end allowance
class TestEndToEndAllowance:
    """oracle.render(slack=...): the per-pixel allowance `derived` must bound what the image of
    ANOTHER record does when that record lies within the stated per-Gaussian slack of this one. Pinned by brute
    force: perturb a record inside its slack (random signs, the worst corner of the box) and render both."""

    def _records(self, seed=3, n=600):
        wl = make_config(0, n=n, seed=seed)
        cam = wl.cameras[0]
        _, rec = oracle.preprocess_scene(wl.scene, cam, 0.37)
        return rec, cam

    def test_zero_slack_changes_nothing(self):
        rec, cam = self._records()
        a = oracle.render(rec, cam.width, cam.height)
        b = oracle.render(rec, cam.width, cam.height, slack=np.zeros((rec.shape[0], 6)))
        assert np.array_equal(a["rgb"], b["rgb"]) and np.array_equal(a["budget"], b["budget"])
        assert np.all(b["derived"] == 0) and np.all(a["derived"] == 0)

    @pytest.mark.parametrize("which", ["mean", "conic", "opacity", "colour", "all"])
    def test_derived_bounds_the_image_of_a_perturbed_record(self, which):
        rec, cam = self._records()
        n = rec.shape[0]
        rng = np.random.default_rng(11)
        live = rec[:, 3] > 0
        sl = np.zeros((n, 6))
        if which in ("mean", "all"):
            sl[:, 0] = sl[:, 1] = 2e-4
        if which in ("conic", "all"):
            sl[:, 2] = 1e-5 * np.sqrt(np.abs(rec[:, 4] * rec[:, 6]))
        if which in ("opacity", "all"):
            sl[:, 3] = 3e-5
        if which in ("colour", "all"):
            sl[:, 4] = 2e-5
        sl[~live] = 0
        base = oracle.render(rec, cam.width, cam.height, slack=sl)
        assert base["derived"].max() > 0
        worst = 0.0
        for trial in range(6):
            sg = rng.choice([-1.0, 1.0], size=(n, 8))
            p = rec.astype(np.float64).copy()
            p[:, 0] += sg[:, 0] * sl[:, 0]
            p[:, 1] += sg[:, 1] * sl[:, 1]
            for j, col in enumerate((4, 5, 6)):
                p[:, col] += sg[:, 2 + j] * sl[:, 2]
            p[:, 3] *= np.exp(sg[:, 5] * sl[:, 3])
            p[:, 8:11] += sg[:, 6:7] * sl[:, 4:5]
            p32 = p.astype(np.float32)
            p32[~live] = rec[~live]
            # the perturbed record is itself rounded to fp32: one more half ulp of every field, far below the slack
            other = oracle.render(p32, cam.width, cam.height)
            err = np.abs(other["rgb"] - base["rgb"]).max(0)
            allow = 1e-7 + base["derived"] + base["budget"]
            assert np.all(err <= allow), (which, trial, float((err - allow).max()))
            ea = np.abs(other["alpha"] - base["alpha"])
            assert np.all(ea <= 1e-7 + (base["derived"] + base["budget"]) / min(1.0, base["c_max"]))
            clean = base["budget"] == 0
            worst = max(worst, float((err[clean] / np.maximum(base["derived"][clean], 1e-30)).max()))
        # the bound is not vacuous: random sign patterns reach a fair share of it
        assert worst > 0.02, worst

    def test_slack_widens_the_cutoff_window(self):
        """A Gaussian whose alpha at a pixel is 1e-3 relative below 1/255 is not fragile on its own, but is once the
        other record's opacity may be 2e-3 higher (it would then pass the cutoff there)."""
        rows = np.stack([record_row(8.5, 8.5, 3.0, (1.0 / 255.0) * (1 - 1e-3), 0.02, 0.0, 0.02)])
        a = oracle.render(rows, 16, 16)
        assert a["budget"][8, 8] == 0
        sl = np.zeros((1, 6))
        sl[0, 3] = 2e-3
        b = oracle.render(rows, 16, 16, slack=sl)
        assert b["budget"][8, 8] > 0

    def test_depth_slack_flags_only_reachable_swaps(self):
        """Two overlapping layers whose depth bits differ by one ulp: with d z = 0 on both the other record visits them
        in the same order (no flag); with d z = 1 ulp on either, a swap is possible and the pixel is flagged with
        alpha_1 alpha_2 T c_max. Equal bits with d z = 0 keep index order on both sides: no flag."""
        z0 = np.float32(3.0)
        z1 = np.nextafter(z0, np.float32(4.0))
        for zb, dz, want in ((z1, 0.0, False), (z1, 1.0, True), (z0, 0.0, False), (np.float32(3.5), 1.0, False)):
            rows = np.stack([record_row(8.5, 8.5, z0, 0.5, 0.02, 0.0, 0.02, rgb=(1, 0, 0)),
                             record_row(8.5, 8.5, zb, 0.5, 0.02, 0.0, 0.02, rgb=(0, 1, 0))])
            sl = np.zeros((2, 6))
            sl[1, 5] = dz
            o = oracle.render(rows, 16, 16, tie_budget=True, slack=sl)
            assert (o["budget"][8, 8] > 0) == want, (zb, dz)
            if want:
                assert np.isclose(o["budget"][8, 8], 0.5 * 0.5 * 1.0 * 1.0)      # = |C(swapped) - C| per channel here
                swapped = rows.copy()
                swapped[0, 2], swapped[1, 2] = rows[1, 2], rows[0, 2]      # the other depth order
                sw = oracle.render(swapped, 16, 16)
                assert np.isclose(np.abs(sw["rgb"][:, 8, 8] - o["rgb"][:, 8, 8]).max(), 0.25)


# ----------------------------------------------------------------------------- exact tile lists (f-4)
class TestExactTiles:
    """P13: only the tiles of a Gaussian's rectangle whose box of pixel centres its region
    { alpha >= 1/255 } can reach are listed. Pinned against brute force in double on the fp32 record:
    safety (no dropped tile has a pixel centre with alpha >= 1/255), kept subset of the rectangle, and tightness
    (kept == 'the box intersects the region', by an independent box-minimum of the quadratic form)."""

    @staticmethod
    def _scenes():
        out = []
        for seed, scale, n in ((0, 1.0, 1500), (5, 4.0, 600), (7, 12.0, 300)):
            wl = make_config(0, n=n, seed=seed)
            s = wl.scene
            sc = one_scene(mu=s.mu, quat=s.quat, scale=s.scale * scale, opacity=s.opacity, sh=s.sh, tau=s.tau, beta=s.beta, vel=s.vel)
            out.append((sc, wl.cameras[0]))
        # needles: one long axis, thin others, random orientations
        rng = np.random.default_rng(3)
        n = 400
        mu = np.stack([rng.uniform(-3, 3, n), rng.uniform(-2, 2, n), rng.uniform(2, 12, n)], 1)
        sc = one_scene(mu=mu, quat=rng.normal(size=(n, 4)), scale=np.stack([rng.uniform(0.5, 3, n), np.full(n, 0.01), np.full(n, 0.01)], 1),
                       opacity=rng.uniform(0.004, 1.0, n))
        out.append((sc, cam_simple(160, 112, 120.0)))
        return out

    @staticmethod
    def _pairs(rec, W, H):
        """(g, tile) pairs of the rectangle list and of the exact list, as sets of g * ntiles + tile."""
        TX, TY = (W + 15) // 16, (H + 15) // 16
        a = oracle.keys(rec, W, H, 0, exact=False)
        b = oracle.keys(rec, W, H, 0, exact=True)
        pa = a["vals_unsorted"].astype(np.int64) * (TX * TY) + (a["keys_unsorted"] >> np.uint64(32)).astype(np.int64)
        pb = b["vals_unsorted"].astype(np.int64) * (TX * TY) + (b["keys_unsorted"] >> np.uint64(32)).astype(np.int64)
        return pa, pb, TX, TY

    @staticmethod
    def _alpha_max_over_pixel_centres(rec, g, tile, TX, W, H):
        r = rec[g].astype(np.float64)
        tx, ty = tile % TX, tile // TX
        xs = np.arange(tx * 16, min(tx * 16 + 16, W)) + 0.5
        ys = np.arange(ty * 16, min(ty * 16 + 16, H)) + 0.5
        dx, dy = np.meshgrid(r[0] - xs, r[1] - ys)
        w = -0.5 * (r[4] * dx * dx + r[6] * dy * dy) - r[5] * dx * dy
        return float((r[3] * np.exp(np.minimum(w, 0.0))).max())

    def test_kept_is_a_subset_and_safe(self):
        dropped_total = 0
        for sc, cam in self._scenes():
            _, rec = P(sc, cam, 0.37)
            pa, pb, TX, TY = self._pairs(rec, cam.width, cam.height)
            sa, sb = set(pa.tolist()), set(pb.tolist())
            assert sb <= sa and len(pb) == len(sb)
            _, c0, M0 = oracle.tile_counts(rec, cam.width, cam.height)
            _, c1, M1 = oracle.tile_counts(rec, cam.width, cam.height, exact=True)
            assert M1 == len(pb) and M0 == len(pa) and np.all(c1 <= c0)
            # (a Gaussian whose region falls between the pixel centres of neighbouring tiles keeps no tile at all)
            for pr in sa - sb:
                g, tile = divmod(pr, TX * TY)
                assert self._alpha_max_over_pixel_centres(rec, g, tile, TX, cam.width, cam.height) < 1.0 / 255.0, (g, tile)
            dropped_total += len(sa - sb)
        assert dropped_total > 500       # the pin bites: many pairs are dropped

    def test_kept_equals_box_intersects_region(self):
        """Independent characterisation: the minimum of q(d) = a dx^2 + 2 b dx dy + c dy^2 over the tile's box of pixel
        centres (0 if the centre is inside, else the least over the four edges of the 1-D quadratic at its clamped
        stationary point), against k = 2 ln(255 o~)."""
        def qmin(r, x0, x1, y0, y1):
            a, b, c = r[4], r[5], r[6]
            dx0, dx1, dy0, dy1 = x0 - r[0], x1 - r[0], y0 - r[1], y1 - r[1]
            if dx0 <= 0 <= dx1 and dy0 <= 0 <= dy1:
                return 0.0
            best = np.inf
            for dx in (dx0, dx1):
                dy = min(max(-b * dx / c, dy0), dy1)
                best = min(best, a * dx * dx + 2 * b * dx * dy + c * dy * dy)
            for dy in (dy0, dy1):
                dx = min(max(-b * dy / a, dx0), dx1)
                best = min(best, a * dx * dx + 2 * b * dx * dy + c * dy * dy)
            return best
        checked = fragile = 0
        for sc, cam in self._scenes():
            _, rec = P(sc, cam, 0.37)
            pa, pb, TX, TY = self._pairs(rec, cam.width, cam.height)
            sb = set(pb.tolist())
            for pr in pa.tolist()[::3]:
                g, tile = divmod(pr, TX * TY)
                r = rec[g].astype(np.float64)
                k = 2.0 * math.log(255.0 * r[3])
                tx, ty = tile % TX, tile // TX
                q = qmin(r, tx * 16 + 0.5, tx * 16 + 15.5, ty * 16 + 0.5, ty * 16 + 15.5)
                # the fp32 test keeps a margin (k (1 + 2e-4) + 2e-5, 1e-3 px); pairs inside that band may go either way
                if abs(q - k) <= 1e-3 * k + 1e-3 + 0.05 * math.sqrt(max(q, k) * max(r[4], r[6])):
                    fragile += 1
                    continue
                assert (pr in sb) == (q <= k), (g, tile, q, k)
                checked += 1
        assert checked > 3000 and fragile < 0.05 * checked

    def test_binned_by_exact_tiles_equals_brute_force(self):
        """The image is the tile-free definition: compositing a pixel over the exact lists must equal compositing it
        over ALL Gaussians, bit for bit in double."""
        for sc, cam in self._scenes()[:2] + self._scenes()[3:]:
            _, rec = P(sc, cam, 0.37)
            a = oracle.render(rec, cam.width, cam.height, mode="brute")
            b = oracle.render(rec, cam.width, cam.height, mode="binned_exact")
            for k in ("rgb", "depth", "alpha"):
                assert np.array_equal(a[k], b[k]), k
            assert b["visited"] < oracle.render(rec, cam.width, cam.height, mode="binned")["visited"]

    def test_lists_ranges_and_single_tile_lists_are_consistent(self):
        sc, cam = self._scenes()[1]
        _, rec = P(sc, cam, 0.37)
        k = oracle.keys(rec, cam.width, cam.height, 1, exact=True)
        assert np.all(np.diff(k["keys_sorted"].astype(np.int64)) >= 0)
        TX, TY = (cam.width + 15) // 16, (cam.height + 15) // 16
        for tile in (0, TX - 1, TX * TY // 2, TX * TY - 1):
            kk, vv = oracle.tile_list(rec, cam.width, cam.height, tile, exact=True)
            b, e = k["ranges"][tile]
            assert np.array_equal(k["vals_sorted"][b:e], vv) and np.array_equal(k["keys_sorted"][b:e], kk)

    def test_special_cases(self):
        cam = cam_simple(128, 96, 100.0)
        # a Gaussian covering the whole image keeps every tile; an isotropic blob keeps a disc, not its square
        big = record_row(64.0, 48.0, 3.0, 0.9, 1e-6, 0.0, 1e-6, hx=float(np.sqrt(2 * math.log(255 * 0.9) / 1e-6)), hy=float(np.sqrt(2 * math.log(255 * 0.9) / 1e-6)))
        _, c0, _ = oracle.tile_counts(big[None], 128, 96)
        _, c1, _ = oracle.tile_counts(big[None], 128, 96, exact=True)
        assert c0[0] == c1[0] == 48
        sig = 12.0
        kq = 2 * math.log(255 * 0.9)
        blob = record_row(64.3, 47.8, 3.0, 0.9, 1 / sig ** 2, 0.0, 1 / sig ** 2, hx=float(sig * math.sqrt(kq)), hy=float(sig * math.sqrt(kq)))
        _, c0, _ = oracle.tile_counts(blob[None], 128, 96)
        _, c1, _ = oracle.tile_counts(blob[None], 128, 96, exact=True)
        assert c1[0] < c0[0]                                  # the corners of the square go
        # at the opacity cutoff (k ~ 0) the region is a point: the Gaussian keeps the tile of its centre
        dot = record_row(40.2, 40.7, 3.0, (1 / 255) * (1 + 1e-6), 0.5, 0.1, 0.5, hx=1e-3, hy=1e-3)
        _, c1, _ = oracle.tile_counts(dot[None], 128, 96, exact=True)
        assert c1[0] == 1
        # a degenerate conic (det <= 0, NaN) keeps the whole rectangle
        for bad in (record_row(60, 40, 3, 0.5, 1e-3, 1e-2, 1e-3, hx=30, hy=30), record_row(60, 40, 3, 0.5, np.nan, 0.0, 1e-3, hx=30, hy=30)):
            _, c0, _ = oracle.tile_counts(bad[None], 128, 96)
            _, c1, _ = oracle.tile_counts(bad[None], 128, 96, exact=True)
            assert c0[0] == c1[0] > 1

    def test_reduction_on_an_urban_shaped_scene(self):
        wl = make_config(2, n=20_000)
        cam = wl.cameras[0]
        _, rec = P(wl.scene, cam, 0.5)
        _, _, M0 = oracle.tile_counts(rec, cam.width, cam.height)
        _, _, M1 = oracle.tile_counts(rec, cam.width, cam.height, exact=True)
        assert M1 < 0.8 * M0, (M0, M1)

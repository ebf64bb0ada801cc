"""Pins of oracle/pilot_footprint.py (supp Eq.2-3) against closed forms on planar heightfields (CPU only)."""
import numpy as np

from oracle import pilot_footprint as pf
from paper_2606_31098_b200 import workloads as wl


def plane_dsm(h0, ax, ay, size=257, gsd=1.0):
    origin = (-(size - 1) * gsd / 2, -(size - 1) * gsd / 2)
    ys, xs = np.mgrid[0:size, 0:size]
    z = h0 + ax * (origin[0] + xs * gsd) + ay * (origin[1] + ys * gsd)
    return z.astype(np.float64), origin, gsd


def ray_plane(C, w, h0, ax, ay):
    # z = h0 + ax x + ay y  <=>  n.p = h0 with n = (-ax, -ay, 1)
    n = np.array([-ax, -ay, 1.0])
    return (h0 - n @ C) / (n @ w)


def test_bilinear_matches_the_refinement_oracle_rule():
    from oracle import pilot_oracle as po
    from tests.small_problems import tiny
    prob = tiny(seed=2)
    b = po.Bound(prob)
    rng = np.random.default_rng(0)
    for _ in range(50):
        x, y = rng.uniform(-40, 40, 2)
        ok, z, _, _ = po.dsm_sample(b, x, y)
        mine = pf.dsm_bilinear(prob["dsm"], prob["dsm_origin"], prob["dsm_gsd"], x, y)
        assert (mine is None) == (not ok)
        if ok:
            assert abs(mine - z) < 1e-12


def test_footprint_on_a_plane_is_the_ray_plane_intersection():
    h0, ax, ay = 12.0, 0.03, -0.02
    dsm, origin, gsd = plane_dsm(h0, ax, ay)
    T = wl.pitched_pose([5.0, -60.0, 90.0], 55.0, 10.0)
    K, W, H = (300.0, 300.0, 159.5, 119.5), 320, 240
    n, s_max = 4000, 400.0
    fp = pf.footprint(T.reshape(-1), K, W, H, dsm, origin, gsd, n, s_max)
    C, rays = pf.corner_rays(T.reshape(-1), K, W, H)
    for c in range(4):
        s_true = ray_plane(C, rays[c], h0, ax, ay)
        assert 0 < s_true < s_max
        s_star = np.linalg.norm(fp[c, :3] - C)
        # on a plane |z_ray - h| is linear in |s - s_true|: the arg-min is the sample nearest to the intersection
        assert abs(s_star - s_true) <= 0.5 * s_max / n + 1e-9
        assert abs(s_star / (s_max / n) - round(s_star / (s_max / n))) < 1e-6        # it IS one of the samples
        slope = abs(rays[c][2] - ax * rays[c][0] - ay * rays[c][1])
        assert abs(fp[c, 3] - slope * abs(s_star - s_true)) < 1e-9
    # the corner order is (0,0), (W-1,0), (W-1,H-1), (0,H-1): top corners look farther than bottom ones
    assert np.linalg.norm(fp[0, :3] - C) > np.linalg.norm(fp[3, :3] - C)
    assert np.linalg.norm(fp[1, :3] - C) > np.linalg.norm(fp[2, :3] - C)


def test_footprint_skips_samples_outside_the_dsm():
    dsm, origin, gsd = plane_dsm(0.0, 0.0, 0.0, size=65)
    T = wl.pitched_pose([0.0, -10.0, 50.0], 20.0)                # shallow: the top rays leave the 64 m map
    fp = pf.footprint(T.reshape(-1), (100.0, 100.0, 31.5, 23.5), 64, 48, dsm, origin, gsd, 500, 1000.0)
    assert np.all(np.isfinite(fp[2:]))                            # bottom corners hit inside
    for c in range(2):                                            # top corners: best sample is the last one inside
        if np.isfinite(fp[c, 0]):
            assert abs(fp[c, 0]) <= 32 and abs(fp[c, 1]) <= 32 and fp[c, 3] > 1.0
    fp = pf.footprint(wl.pitched_pose([500.0, 500.0, 50.0], 45.0).reshape(-1), (100.0, 100.0, 31.5, 23.5), 64, 48,
                      dsm, origin, gsd, 100, 100.0)
    assert np.all(np.isnan(fp))                                   # a camera far off the map: no footprint


def test_homography_properties():
    rng = np.random.default_rng(3)
    quad = np.array([[-40.0, 80.0], [55.0, 90.0], [30.0, -20.0], [-25.0, -15.0]])
    Wc, Hc = 128, 96
    Hm = pf.homography(quad, Wc, Hc)
    src = np.array([[0, 0, 1], [Wc - 1, 0, 1], [Wc - 1, Hc - 1, 1], [0, Hc - 1, 1.0]])
    q = (Hm @ src.T).T
    assert np.allclose(q[:, :2] / q[:, 2:], quad, atol=1e-9)      # its four defining correspondences
    for _ in range(10):                                           # projective maps preserve collinearity
        a, b = rng.uniform(0, 95, 2), rng.uniform(0, 95, 2)
        pts = np.array([a, b, 0.3 * a + 0.7 * b])
        m = (Hm @ np.c_[pts, np.ones(3)].T).T
        m = m[:, :2] / m[:, 2:]
        d1, d2 = m[1] - m[0], m[2] - m[0]
        assert abs(d1[0] * d2[1] - d1[1] * d2[0]) < 1e-8
    # a parallelogram footprint: the homography is affine (bottom row (0, 0, 1)), the centre maps to the centroid
    para = np.array([[0.0, 0.0], [10.0, 2.0], [13.0, 9.0], [3.0, 7.0]])
    Ha = pf.homography(para, 11, 21)
    assert np.allclose(Ha[2], [0, 0, 1], atol=1e-12)
    c = Ha @ np.array([5.0, 10.0, 1.0])
    assert np.allclose(c[:2] / c[2], para.mean(0))


def test_lifted_anchors_on_a_plane_are_the_back_projected_pixels():
    """Over a planar DSM the map from image pixels to the ground is a homography, so — with the crop sized like the
    image — the anchor of crop pixel (u, v) must be the ray/plane intersection of image pixel (u, v) (supp Eq.3)."""
    h0, ax, ay = 7.0, 0.02, 0.015
    dsm, origin, gsd = plane_dsm(h0, ax, ay, size=513, gsd=1.0)
    T = wl.pitched_pose([-8.0, -70.0, 95.0], 50.0, -15.0)
    K, W, H = (280.0, 290.0, 150.0, 110.0), 320, 240
    C, rays = pf.corner_rays(T.reshape(-1), K, W, H)
    # exact footprint (not the sampled one) so that the pin isolates the homography + lift
    corners = np.array([np.append(C + ray_plane(C, r, h0, ax, ay) * r, 0.0) for r in rays])
    rng = np.random.default_rng(4)
    pix = rng.uniform([0, 0], [W - 1, H - 1], (200, 2))
    anchors = pf.lift_anchors(corners, W, H, pix, dsm, origin, gsd)
    R = T[:, :3]
    for (u, v), P in zip(pix, anchors):
        d = R @ np.array([(u - K[2]) / K[0], (v - K[3]) / K[1], 1.0])
        p = C + ray_plane(C, d, h0, ax, ay) * d
        assert P[3] == 1.0 and np.allclose(P[:3], p, atol=1e-8)
    # outside the DSM: weight 0
    far = pf.lift_anchors(corners + [1e4, 0, 0, 0], W, H, pix[:3], dsm, origin, gsd)
    assert np.all(far[:, 3] == 0) and np.all(far[:, 2] == 0)

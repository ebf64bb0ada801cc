"""Pins of oracle/pilot_supervision.py (supp Eq.7-8) against closed forms. CPU only."""
import numpy as np
import pytest

from oracle import pilot_supervision as ps


def test_barron_named_special_cases():
    s = np.array([0.0, 1e-3, 0.5, 2.0, 37.0])
    c = 1.7
    z = s / c ** 2
    assert np.allclose(ps.barron_rho(s, 2.0, c), 0.5 * z, rtol=1e-14)                         # L2
    assert np.allclose(ps.barron_rho(s, 1.0, c), np.sqrt(z + 1.0) - 1.0, rtol=1e-12)           # Charbonnier / pseudo-Huber
    assert np.allclose(ps.barron_rho(s, 0.0, c), np.log(0.5 * z + 1.0), rtol=1e-12)            # Cauchy
    assert np.allclose(ps.barron_rho(s, -2.0, c), 2.0 * z / (z + 4.0), rtol=1e-12)             # Geman-McClure
    assert np.allclose(ps.barron_rho(s, -np.inf, c), 1.0 - np.exp(-0.5 * z), rtol=1e-12)       # Welsch


def test_barron_is_continuous_at_its_removable_singularities_and_monotone():
    s = np.linspace(0.0, 25.0, 51)
    for a0 in (0.0, 2.0):
        lim = ps.barron_rho(s, a0, 1.3)
        for eps in (1e-6, -1e-6):
            assert np.allclose(ps.barron_rho(s, a0 + eps, 1.3), lim, rtol=1e-4, atol=1e-9)
    assert np.allclose(ps.barron_rho(s, -1e7, 1.3), ps.barron_rho(s, -np.inf, 1.3), rtol=1e-5, atol=1e-9)
    for a in (2.0, 1.0, 0.0, -2.0, -np.inf, 0.5, -7.0):
        r = ps.barron_rho(s, a, 1.3)
        assert r[0] == 0.0 and np.all(np.diff(r) > 0.0)
    # small residuals: every shape is quadratic, rho -> z / 2
    tiny = np.array([1e-8])
    for a in (1.0, 0.0, -2.0, -np.inf, 0.5):
        assert np.allclose(ps.barron_rho(tiny, a, 1.0), 0.5 * tiny, rtol=1e-6)


def _scene(seed=3, n=500):
    rng = np.random.default_rng(seed)
    pts = np.column_stack([rng.uniform(-40, 40, n), rng.uniform(-30, 30, n), rng.uniform(60, 90, n), np.ones(n)])
    pose = np.hstack([np.eye(3), np.zeros((3, 1))]).reshape(12)           # camera at the origin looking along +z
    K = (400.0, 400.0, 320.0, 240.0)
    return pts, pose, K


def test_loss_is_zero_at_the_ground_truth_pose():
    pts, pose, K = _scene()
    L, n = ps.reprojection_loss(pose[None], pose, pts, K, 640, 480, 0.1, 1.0, 2.0)
    assert L[0] == 0.0 and 0 < n[0] <= len(pts)


def test_roll_about_the_optical_axis_closed_form():
    pts, pose, K = _scene()
    th = 0.07
    Rz = np.array([[np.cos(th), -np.sin(th), 0.0], [np.sin(th), np.cos(th), 0.0], [0.0, 0.0, 1.0]])
    rolled = np.hstack([Rz, np.zeros((3, 1))]).reshape(12)
    us, vs, zs = ps.project(pose, pts, K)
    vis = (zs > 0.1) & (us >= 0) & (vs >= 0) & (us <= 639) & (vs <= 479)
    s = 2.0 * (1.0 - np.cos(th)) * ((us[vis] - K[2]) ** 2 + (vs[vis] - K[3]) ** 2)
    for alpha in (2.0, 1.0, 0.0, -2.0):
        L, n = ps.reprojection_loss(rolled[None], pose, pts, K, 640, 480, 0.1, alpha, 3.0)
        assert n[0] == vis.sum()
        assert L[0] == pytest.approx(np.mean(ps.barron_rho(s, alpha, 3.0)), rel=1e-10)


def test_sideways_shift_over_a_fronto_parallel_plane():
    rng = np.random.default_rng(5)
    n, Z, t = 300, 75.0, 1.25
    pts = np.column_stack([rng.uniform(-30, 30, n), rng.uniform(-20, 20, n), np.full(n, Z), np.ones(n)])
    pose = np.hstack([np.eye(3), np.zeros((3, 1))]).reshape(12)
    moved = np.hstack([np.eye(3), np.array([[t], [0.0], [0.0]])]).reshape(12)
    K = (400.0, 400.0, 320.0, 240.0)
    L, cnt = ps.reprojection_loss(moved[None], pose, pts, K, 640, 480, 0.1, 2.0, 1.0)
    assert cnt[0] == n                                             # all inside the image by construction
    assert L[0] == pytest.approx(0.5 * (K[0] * t / Z) ** 2, rel=1e-12)


def test_visible_set_and_empty_set():
    pts, pose, K = _scene()
    behind = pts.copy(); behind[:, 2] = -behind[:, 2]
    L, n = ps.reprojection_loss(pose[None], pose, behind, K, 640, 480, 0.1, 1.0, 1.0)
    assert n[0] == 0 and L[0] == 0.0
    # a point in front of the ground-truth camera but behind the optimised one leaves V
    far = np.hstack([np.eye(3), np.array([[0.0], [0.0], [200.0]])]).reshape(12)
    L, n = ps.reprojection_loss(far[None], pose, pts, K, 640, 480, 0.1, 1.0, 1.0)
    assert n[0] == 0

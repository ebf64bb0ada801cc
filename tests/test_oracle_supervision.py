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


# ------------------------------------------------------------------ backward pieces, pinned by central differences

def _xi_mat(xi):
    M = np.zeros((4, 4))
    M[:3, :3] = [[0, -xi[5], xi[4]], [xi[5], 0, -xi[3]], [-xi[4], xi[3], 0]]
    M[:3, 3] = xi[:3]
    return M


def _T_cw(pose):
    T = np.asarray(pose, np.float64).reshape(3, 4)
    M = np.eye(4); M[:3, :3] = T[:, :3].T; M[:3, 3] = -T[:, :3].T @ T[:, 3]
    return M


def _pose_of(M):
    R_wc = M[:3, :3].T
    return np.concatenate([R_wc, (-R_wc @ M[:3, 3])[:, None]], 1).reshape(-1)


def _bscene(seed=5, n=300):
    rng = np.random.default_rng(seed)
    pts = np.concatenate([rng.uniform(-40, 40, (n, 2)), rng.uniform(0, 10, (n, 1)), np.ones((n, 1))], 1)
    from tests.small_problems import look_down_pose
    Ts = look_down_pose(np.array([0.0, -60.0, 100.0])).reshape(-1)
    K = (300.0, 310.0, 160.0, 120.0)
    return pts, Ts, K


def test_loss_gradient_matches_central_differences_of_the_forward_value():
    from scipy.linalg import expm
    pts, Ts, K = _bscene()
    Tk = _pose_of(expm(_xi_mat(np.array([1.5, -2.0, 0.8, 0.02, -0.015, 0.03]))) @ _T_cw(Ts))
    for alpha, c in [(2.0, 1.0), (1.0, 3.0), (0.0, 2.0), (-2.0, 4.0), (-np.inf, 5.0), (0.5, 2.5)]:
        L, n, G = ps.reprojection_loss_grad(Tk[None], Ts, pts, K, 320, 240, 0.1, alpha, c)
        L0, n0 = ps.reprojection_loss(Tk[None], Ts, pts, K, 320, 240, 0.1, alpha, c)
        assert L[0] == L0[0] and n[0] == n0[0] and n[0] > 100
        for i in range(6):
            e = np.zeros(6); e[i] = 1e-6
            Lp = ps.reprojection_loss(_pose_of(expm(_xi_mat(e)) @ _T_cw(Tk))[None], Ts, pts, K, 320, 240, 0.1, alpha, c)[0][0]
            Lm = ps.reprojection_loss(_pose_of(expm(_xi_mat(-e)) @ _T_cw(Tk))[None], Ts, pts, K, 320, 240, 0.1, alpha, c)[0][0]
            assert (Lp - Lm) / 2e-6 == pytest.approx(G[0, i], rel=2e-6, abs=1e-9 * np.abs(G[0]).max()), (alpha, i)
    # at the ground truth the loss is stationary
    assert np.allclose(ps.reprojection_loss_grad(Ts[None], Ts, pts, K, 320, 240, 0.1, 1.0, 2.0)[2], 0.0, atol=1e-15)


def test_left_jacobian_defining_property():
    from scipy.linalg import expm, logm
    rng = np.random.default_rng(8)
    for scale in (1e-3, 0.2, 1.0):
        xi = rng.normal(size=6) * scale
        J = ps.se3_left_jacobian(xi)
        for i in range(6):
            d = np.zeros(6); d[i] = 1e-6
            Lg = np.real(logm(expm(_xi_mat(xi + d)) @ np.linalg.inv(expm(_xi_mat(xi)))))     # exp((J_l d)^) to first order
            col = np.array([Lg[0, 3], Lg[1, 3], Lg[2, 3], Lg[2, 1], Lg[0, 2], Lg[1, 0]]) / 1e-6
            assert np.allclose(col, J[:, i], atol=5e-6 * max(1.0, scale))
    assert np.allclose(ps.se3_left_jacobian(np.zeros(6)), np.eye(6))
    xi = rng.normal(size=6) * 0.3
    assert np.allclose(ps.se3_exp_matrix(xi), expm(_xi_mat(xi)), atol=1e-13)


@pytest.mark.parametrize("diag", [False, True])
def test_lm_step_adjoint_matches_central_differences_of_the_composed_map(diag):
    """f(H, g, eps) = L(exp(dxi(H, g)^) exp(eps^) T^k): dL/dg, dL/dH (symmetric perturbations) and q_prev = df/d eps."""
    from scipy.linalg import expm
    pts, Ts, K = _bscene(seed=6)
    rng = np.random.default_rng(11)
    Tk = expm(_xi_mat(np.array([2.0, 1.0, -1.5, -0.02, 0.03, 0.01]))) @ _T_cw(Ts)
    B = rng.normal(size=(12, 6)) * np.array([1, 1, 1, 30, 30, 30])
    Hm = B.T @ B
    g = rng.normal(size=6) * np.array([1.0, 1.0, 1.0, 40.0, 40.0, 40.0])
    lam = 0.3 if diag else 5.0
    al, c = 1.0, 3.0

    def step(Hm, g):
        D = np.diag(np.maximum(np.diag(Hm), 1e-12)) if diag else np.eye(6)
        return -np.linalg.solve(Hm + lam * D, g)

    def f(Hm, g, eps=np.zeros(6)):
        T = expm(_xi_mat(step(Hm, g))) @ expm(_xi_mat(eps)) @ Tk
        return ps.reprojection_loss(_pose_of(T)[None], Ts, pts, K, 320, 240, 0.1, al, c)[0][0]

    dxi0 = step(Hm, g)
    assert 0.05 < np.linalg.norm(dxi0[:3]) < 5 and np.linalg.norm(dxi0[3:]) > 1e-3      # a step large enough for J_l to matter
    T1 = _pose_of(expm(_xi_mat(dxi0)) @ Tk)
    q = ps.reprojection_loss_grad(T1[None], Ts, pts, K, 320, 240, 0.1, al, c)[2][0]
    dxi, GH, Gg, qp = ps.lm_step_adjoint(Hm, g, lam, diag, q)
    assert np.allclose(dxi, dxi0)
    scale_g = np.abs(Gg).max()
    for i in range(6):
        h = 1e-5 * max(1.0, abs(g[i]))
        e = np.zeros(6); e[i] = h
        assert (f(Hm, g + e) - f(Hm, g - e)) / (2 * h) == pytest.approx(Gg[i], rel=1e-5, abs=1e-7 * scale_g)
    scale_H = np.abs(GH).max()
    for i in range(6):
        for j in range(i, 6):
            h = 1e-5 * max(1.0, abs(Hm[i, j]))
            E = np.zeros((6, 6)); E[i, j] = E[j, i] = h
            fd = (f(Hm + E, g) - f(Hm - E, g)) / (2 * h)
            want = GH[i, j] if i == j else 2 * GH[i, j]            # dL = <G_H, dH>: an off-diagonal pair is perturbed together
            assert fd == pytest.approx(want, rel=2e-5, abs=1e-6 * scale_H), (i, j)
    for i in range(6):
        e = np.zeros(6); e[i] = 1e-6
        assert (f(Hm, g, e) - f(Hm, g, -e)) / 2e-6 == pytest.approx(qp[i], rel=1e-5, abs=1e-8 * np.abs(qp).max())

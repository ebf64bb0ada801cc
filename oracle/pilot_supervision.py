"""CPU ORACLE of the unrolled reprojection supervision, forward value and backward pieces (numpy, float64).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module. It shares no code with paper_2606_31098_b200/csrc.

Passages followed (arxiv/paper_2606_31098, supp III-C, PAPER.md line numbers):
  * p*_j = pi(K, T* P_j), p^k_j = pi(K, T^k P_j): ground-truth and optimised projection of a sampled 3D point
    (supp Eq.7); poses are given as the paper's camera-to-world [R_wc | C], so T P = R_wc^T (P - C)
  * L_k = 1/|V| sum_{j in V} rho_B(||p^k_j - p*_j||_2^2), V the visible point set, rho_B the Barron robust loss
    (supp Eq.8).
The general robust loss (Barron, CVPR 2019, the paper's reference [3]) on a squared residual s with shape alpha and
scale c, z = s / c^2:   rho = |alpha-2|/alpha * ((z/|alpha-2| + 1)^(alpha/2) - 1), with the limits
alpha = 2: z/2;  alpha = 0: log(z/2 + 1);  alpha = -inf: 1 - exp(-z/2).
Readings where the paper is silent (A23): alpha and c are parameters (the paper gives neither);
V = points in front of BOTH cameras (Z > z_near) whose GROUND-TRUTH projection lies inside [0, W-1] x [0, H-1] — the
optimised projection may leave the image and must still be penalised; an empty V gives L = 0 and n = 0.

Backward pieces of the unrolled refinement ("the refinement is unrolled"), each the plain
derivative written out:
  * reprojection_loss_grad: dL_k/d eps for the left perturbation T_cw <- exp(eps^) T_cw of the optimised pose (the LM's own
    parametrisation, reading A1/A2: eps = (rho; phi)): 1/|V| sum rho_B'(s_j) 2 (p_j - p_j*)^T J_uv(j), J_uv the 2x6
    projection Jacobian of Eq.(8)'s linearisation;
  * lm_step_adjoint: one LM step dxi = -(H + lambda D)^-1 g (Eq.8), T' = exp(dxi^) T (Eq.9), read
    backwards: given q = dL/d eps' at the UPDATED pose it returns dL/dg, dL/dH (symmetric, so that dL = <G_H, dH> for
    symmetric dH) and the part of dL/d eps at the previous pose that flows through the retraction. With A = H + lambda D:
    v = J_l(dxi)^T q (J_l the left Jacobian of SE(3): exp((xi + d)^) = exp((J_l d)^) exp(xi^) to first order, the textbook
    series sum_n ad(xi)^n / (n+1)!), w = -A^-1 v, dL/dg = w, dL/dH = sym(w dxi^T) [+ lambda diag(w . dxi) for DAMP_DIAG],
    q_prev = Ad(exp(dxi^))^T q. What is NOT here: the dependence of H and g on the previous pose and on the feature maps
    (the transpose of the gather), which needs training data to mean anything.

Pins of the backward pieces (tests/test_oracle_supervision.py): central differences of the forward functions above with the
perturbations built from scipy.linalg.expm in the test (loss gradient; dL/dg, dL/dH and q_prev through the composed map
(H, g, T) -> L(exp(dxi(H, g)^) T)); J_l against its defining property with expm / logm.

Pins (tests/test_oracle_supervision.py): the named special cases of the general loss in closed form (alpha = 2, 1, 0, -2,
-inf), continuity around the removable singularities, monotonicity; L = 0 at T^k = T*; a roll of theta about the optical
axis moves every projection on a circle about the principal point (fx = fy): ||p - p*||^2 = 2 (1 - cos theta) ||p* - c||^2;
a fronto-parallel plane under a sideways camera shift t: every point moves by fx * t / Z.
"""
import numpy as np


def barron_rho(s, alpha, c):
    """General robust loss on the squared residual s >= 0 (array), shape alpha (float, may be -inf), scale c > 0."""
    z = np.asarray(s, np.float64) / (float(c) * float(c))
    if alpha == 2.0:
        return 0.5 * z
    if alpha == 0.0:
        return np.log1p(0.5 * z)
    if alpha == -np.inf:
        return -np.expm1(-0.5 * z)
    b = abs(alpha - 2.0)
    return (b / alpha) * (np.power(z / b + 1.0, 0.5 * alpha) - 1.0)


def project(pose, points, K):
    """pi(K, T P) for pose = [R_wc | C] (12 values, row-major 3x4): returns (u, v, Z) arrays."""
    T = np.asarray(pose, np.float64).reshape(3, 4)
    P = np.asarray(points, np.float64)[:, :3]
    pc = (P - T[:, 3]) @ T[:, :3]                       # rows: R_wc^T (P - C)
    fx, fy, cx, cy = [float(k) for k in K]
    with np.errstate(divide="ignore", invalid="ignore"):
        u = fx * pc[:, 0] / pc[:, 2] + cx
        v = fy * pc[:, 1] / pc[:, 2] + cy
    return u, v, pc[:, 2]


def reprojection_loss(poses, pose_star, points, K, width, height, z_near, alpha, c):
    """supp Eq.(8) for every pose of poses [n][12]. Returns (L [n], |V| [n])."""
    poses = np.asarray(poses, np.float64).reshape(-1, 12)
    us, vs, zs = project(pose_star, points, K)
    ok_star = (zs > z_near) & (us >= 0.0) & (vs >= 0.0) & (us <= width - 1.0) & (vs <= height - 1.0)
    L = np.zeros(len(poses))
    n = np.zeros(len(poses), np.int64)
    for k, pose in enumerate(poses):
        u, v, z = project(pose, points, K)
        vis = ok_star & (z > z_near)
        n[k] = int(vis.sum())
        if n[k]:
            s = (u[vis] - us[vis]) ** 2 + (v[vis] - vs[vis]) ** 2
            L[k] = float(np.sum(barron_rho(s, alpha, c))) / n[k]
    return L, n


# ------------------------------------------------------------------ backward pieces

def barron_drho(s, alpha, c):
    """d rho / d s of the general robust loss (s the squared residual)."""
    c2 = float(c) * float(c)
    z = np.asarray(s, np.float64) / c2
    if alpha == 2.0:
        return np.full(z.shape, 0.5 / c2)
    if alpha == 0.0:
        return 0.5 / (1.0 + 0.5 * z) / c2
    if alpha == -np.inf:
        return 0.5 * np.exp(-0.5 * z) / c2
    b = abs(alpha - 2.0)
    return 0.5 * np.power(z / b + 1.0, 0.5 * alpha - 1.0) / c2


def hat(a):
    return np.array([[0.0, -a[2], a[1]], [a[2], 0.0, -a[0]], [-a[1], a[0], 0.0]])


def reprojection_loss_grad(poses, pose_star, points, K, width, height, z_near, alpha, c):
    """(L [n], |V| [n], dL/d eps [n][6]) with eps = (rho; phi) the left perturbation of T_cw = [R_wc^T | -R_wc^T C]."""
    poses = np.asarray(poses, np.float64).reshape(-1, 12)
    fx, fy = float(K[0]), float(K[1])
    us, vs, zs = project(pose_star, points, K)
    ok_star = (zs > z_near) & (us >= 0.0) & (vs >= 0.0) & (us <= width - 1.0) & (vs <= height - 1.0)
    L, n, G = np.zeros(len(poses)), np.zeros(len(poses), np.int64), np.zeros((len(poses), 6))
    P = np.asarray(points, np.float64)[:, :3]
    for k, pose in enumerate(poses):
        T = pose.reshape(3, 4)
        pc = (P - T[:, 3]) @ T[:, :3]
        u, v, z = project(pose, points, K)
        vis = ok_star & (z > z_near)
        n[k] = int(vis.sum())
        if not n[k]:
            continue
        du, dv = u[vis] - us[vis], v[vis] - vs[vis]
        s = du * du + dv * dv
        L[k] = float(np.sum(barron_rho(s, alpha, c))) / n[k]
        X, Y, Z = pc[vis, 0], pc[vis, 1], pc[vis, 2]
        Ju = np.stack([fx / Z, 0 * Z, -fx * X / Z ** 2, -fx * X * Y / Z ** 2, fx * (1 + X * X / Z ** 2), -fx * Y / Z], 1)
        Jv = np.stack([0 * Z, fy / Z, -fy * Y / Z ** 2, -fy * (1 + Y * Y / Z ** 2), fy * X * Y / Z ** 2, fy * X / Z], 1)
        wgt = 2.0 * barron_drho(s, alpha, c)
        G[k] = ((wgt * du)[:, None] * Ju + (wgt * dv)[:, None] * Jv).sum(0) / n[k]
    return L, n, G


def se3_ad(xi):
    """ad(xi) for xi = (rho; phi): [[phi^, rho^], [0, phi^]]."""
    A = np.zeros((6, 6))
    A[:3, :3] = hat(xi[3:]); A[:3, 3:] = hat(xi[:3]); A[3:, 3:] = hat(xi[3:])
    return A


def se3_left_jacobian(xi, terms=30):
    """J_l(xi) = sum_{n>=0} ad(xi)^n / (n+1)! (the series, written out)."""
    A = se3_ad(np.asarray(xi, np.float64))
    J, term = np.eye(6), np.eye(6)
    for n in range(1, terms):
        term = term @ A / (n + 1)
        J = J + term
    return J


def se3_exp_matrix(xi):
    """exp(xi^) as a 4x4 matrix by its power series (the definition)."""
    M = np.zeros((4, 4))
    M[:3, :3] = hat(xi[3:]); M[:3, 3] = xi[:3]
    E, term = np.eye(4), np.eye(4)
    for n in range(1, 40):
        term = term @ M / n
        E = E + term
    return E


def se3_Ad(T):
    """Ad(T) for T = [[E, t], [0, 1]] in the (rho; phi) ordering: [[E, t^ E], [0, E]]."""
    E, t = T[:3, :3], T[:3, 3]
    A = np.zeros((6, 6))
    A[:3, :3] = E; A[:3, 3:] = hat(t) @ E; A[3:, 3:] = E
    return A


def lm_step_adjoint(Hm, g, lam, damp_diag, q):
    """One LM step read backwards. Hm [6][6] symmetric, g [6], lam scalar, q = dL/d eps at the updated pose.
    Returns (dxi, dL/dH [6][6] symmetric, dL/dg [6], q_prev [6])."""
    Hm, g, q = np.asarray(Hm, np.float64).reshape(6, 6), np.asarray(g, np.float64), np.asarray(q, np.float64)
    D = np.diag(np.maximum(np.diag(Hm), 1e-12)) if damp_diag else np.eye(6)
    A = Hm + lam * D
    dxi = -np.linalg.solve(A, g)
    v = se3_left_jacobian(dxi).T @ q
    w = -np.linalg.solve(A, v)
    GH = 0.5 * (np.outer(w, dxi) + np.outer(dxi, w))
    if damp_diag:
        GH = GH + lam * np.diag(w * dxi * (np.diag(Hm) > 1e-12))
    q_prev = se3_Ad(se3_exp_matrix(dxi)).T @ q
    return dxi, GH, w, q_prev

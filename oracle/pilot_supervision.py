"""CPU ORACLE of the unrolled reprojection supervision, forward value only (numpy, float64).

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
optimised projection may leave the image and must still be penalised; an empty V gives L = 0 and n = 0. Only the
forward value is built: the backward pass through the unrolled LM steps needs training data that is not here.

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

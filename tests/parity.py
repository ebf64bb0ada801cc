"""GPU-vs-oracle comparison helpers (SURVEY.md §8(c) parity protocol)."""
import numpy as np


def level_slice(prob, l, poses=None, iters=1):
    """Single-level problem made of level l of `prob` (teacher-forced evaluation at `poses`)."""
    q = dict(prob)
    q["n_levels"] = 1
    for k in ("width", "height", "channels", "query_feat", "intrinsics", "points", "ref_feat"):
        q[k] = [prob[k][l]]
    q["query_conf"] = [prob.get("query_conf", [None] * prob["n_levels"])[l]]
    if poses is not None:
        q["init_poses"] = np.ascontiguousarray(poses, np.float32).reshape(-1, 12)
    P = dict(prob.get("params", {}))
    P["iters"] = [iters]
    q["params"] = P
    return q


def rot_angle(Ta, Tb):
    """Angle (rad) between the rotations of two [.., 12] poses."""
    Ra = np.asarray(Ta, np.float64).reshape(-1, 3, 4)[:, :, :3]
    Rb = np.asarray(Tb, np.float64).reshape(-1, 3, 4)[:, :, :3]
    D = np.einsum("nij,nik->njk", Ra, Rb)
    # robust small-angle: |log(D)| from the skew part and the trace
    s = 0.5 * np.sqrt((D[:, 2, 1] - D[:, 1, 2]) ** 2 + (D[:, 0, 2] - D[:, 2, 0]) ** 2 + (D[:, 1, 0] - D[:, 0, 1]) ** 2)
    c = 0.5 * (np.trace(D, axis1=1, axis2=2) - 1)
    return np.arctan2(s, c)


def trans_dist(Ta, Tb):
    Ca = np.asarray(Ta, np.float64).reshape(-1, 3, 4)[:, :, 3]
    Cb = np.asarray(Tb, np.float64).reshape(-1, 3, 4)[:, :, 3]
    return np.linalg.norm(Ca - Cb, axis=1)


def system_errors(gpu, orc, rec=0):
    """Per-hypothesis relative errors of the recorded system `rec`: H (Frobenius), g (vs g_abs), cost."""
    Hg, Ho = gpu["iter_hessian"][rec].astype(np.float64), orc["iter_hessian"][rec].astype(np.float64)
    gg, go = gpu["iter_gradient"][rec].astype(np.float64), orc["iter_gradient"][rec].astype(np.float64)
    cg, co = gpu["iter_cost"][rec].astype(np.float64), orc["iter_cost"][rec].astype(np.float64)
    eH = np.linalg.norm(Hg - Ho, axis=1) / np.maximum(np.linalg.norm(Ho, axis=1), 1e-300)
    eg = np.linalg.norm(gg - go, axis=1) / np.maximum(orc["iter_gabs"][rec], 1e-300)
    both_inf = np.isinf(cg) & np.isinf(co)
    ec = np.where(both_inf, 0.0, np.abs(cg - co) / np.maximum(np.abs(co), 1e-300))
    return eH, eg, ec


def converged(orc, step_tol=1e-5):
    return (orc["last_step"] < step_tol) & np.isfinite(orc["cost64"])


def pose_errors(gpu, orc):
    return rot_angle(gpu["poses"], orc["poses64"]), trans_dist(gpu["poses"], orc["poses64"])


from paper_2606_31098_b200.workloads import levels_slice  # noqa: E402,F401  (dict slicing; lives with the generators)

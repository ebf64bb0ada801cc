"""Pins of oracle/pilot_photo_backward.py: central differences of the C oracle's pilot_oracle_eval (photo term only, the
forward definition) with respect to map entries, reference entries and the pose. CPU only."""
import numpy as np
import pytest
from scipy.linalg import expm

from oracle import pilot_oracle as po
from oracle import pilot_photo_backward as pb
from tests.small_problems import tiny


def _xi_mat(xi):
    M = np.zeros((4, 4))
    M[:3, :3] = [[0, -xi[5], xi[4]], [xi[5], 0, -xi[3]], [-xi[4], xi[3], 0]]
    M[:3, 3] = xi[:3]
    return M


def _perturb(pose, eps):
    T = np.asarray(pose, np.float64).reshape(3, 4)
    M = np.eye(4); M[:3, :3] = T[:, :3].T; M[:3, 3] = -T[:, :3].T @ T[:, 3]
    M = expm(_xi_mat(eps)) @ M
    R_wc = M[:3, :3].T
    return np.concatenate([R_wc, (-R_wc @ M[:3, 3])[:, None]], 1).reshape(-1)


def _S(prob, params, pose, GH, Gg):
    """<G_H, H> + <G_g, g> from the forward oracle (photo term only: which = 1)."""
    ev = po.evaluate(po.Bound(prob, params), 0, *po.pose_to_RC(pose), which=1)
    return float(np.sum(GH * ev["H"]) + Gg @ ev["g"])


@pytest.mark.parametrize("loss,scale,conf", [("l2", 0.0, False), ("huber", 0.25, False), ("cauchy", 0.3, True), ("huber", 0.25, True)])
def test_backward_matches_central_differences_of_the_forward_oracle(loss, scale, conf):
    prob = tiny(seed=41, N=25, C=3, conf=conf)
    prob["query_feat"] = [prob["query_feat"][0].astype(np.float64).astype(np.float32)]
    rng = np.random.default_rng(7)
    B = rng.normal(size=(6, 6)); GH = B + B.T
    Gg = rng.normal(size=6)
    params = dict(loss=loss, loss_scale=scale, min_valid=1, w_gravity=0.0, range_mode="off")
    pose = _perturb(prob["gt_pose"], np.array([0.3, -0.2, 0.4, 0.004, -0.003, 0.005]))
    qc = prob["query_conf"][0] if conf else None
    K32 = [float(np.float32(k)) for k in prob["K"]]          # the C-ABI carries the intrinsics as fp32
    dF, dref, deps, S, dconf = pb.photo_backward(prob["query_feat"][0], prob["ref_feat"][0], prob["points"][0], pose, K32, GH, Gg,
                                          loss, float(np.float32(scale)), float(np.float32(0.1)), qc)
    assert S == pytest.approx(_S(prob, params, pose, GH, Gg), rel=1e-10)
    assert np.count_nonzero(np.abs(dF).sum(-1)) >= 30
    # map entries: the strongest ones and a few random touched ones; steps exactly representable in fp32
    F0 = prob["query_feat"][0]
    idx = np.argwhere(np.abs(dF) > 0)
    order = np.argsort(-np.abs(dF[tuple(idx.T)]))
    pick = list(order[:6]) + list(rng.choice(len(idx), 6, replace=False))
    h = 2.0 ** -7
    for k in pick:
        y, x, c = idx[k]
        vals = []
        for sgn in (+1, -1):
            Fp = F0.copy(); Fp[y, x, c] = np.float32(F0[y, x, c] + sgn * h)
            q = dict(prob); q["query_feat"] = [Fp]
            vals.append(_S(q, params, pose, GH, Gg))
        step = float(np.float32(F0[y, x, c] + h)) - float(np.float32(F0[y, x, c] - h))
        fd = (vals[0] - vals[1]) / step
        assert fd == pytest.approx(dF[y, x, c], rel=3e-3, abs=2e-4 * np.abs(dF).max()), (y, x, c)   # S is quadratic+ in F: O(h^2)
    # reference entries
    r0 = prob["ref_feat"][0]
    for j, c in [(int(i), int(k)) for i, k in zip(rng.integers(0, 25, 6), rng.integers(0, 3, 6))]:
        if not np.any(dref[j]):
            continue
        vals = []
        for sgn in (+1, -1):
            rp = r0.copy(); rp[j, c] = np.float32(r0[j, c] + sgn * h)
            q = dict(prob); q["ref_feat"] = [rp]
            vals.append(_S(q, params, pose, GH, Gg))
        step = float(np.float32(r0[j, c] + h)) - float(np.float32(r0[j, c] - h))
        assert (vals[0] - vals[1]) / step == pytest.approx(dref[j, c], rel=3e-3, abs=2e-4 * np.abs(dref).max()), (j, c)
    # confidence map entries
    if conf:
        q0 = prob["query_conf"][0]
        idq = np.argwhere(np.abs(dconf) > 0)
        for k in rng.choice(len(idq), 6, replace=False):
            y, x = idq[k]
            vals = []
            for sgn in (+1, -1):
                qp = q0.copy(); qp[y, x] = np.float32(q0[y, x] + sgn * h)
                qq = dict(prob); qq["query_conf"] = [qp]
                vals.append(_S(qq, params, pose, GH, Gg))
            step = float(np.float32(q0[y, x] + h)) - float(np.float32(q0[y, x] - h))
            assert (vals[0] - vals[1]) / step == pytest.approx(dconf[y, x], rel=3e-3, abs=2e-4 * np.abs(dconf).max()), (y, x)
    else:
        assert dconf is None
    # pose: six directions of the left perturbation (small steps: the bilinear cells must not change)
    for i in range(6):
        e = np.zeros(6); e[i] = 1e-6 if i < 3 else 1e-8
        fd = (_S(prob, params, _perturb(pose, e), GH, Gg) - _S(prob, params, _perturb(pose, -e), GH, Gg)) / (2 * e[i])
        assert fd == pytest.approx(deps[i], rel=2e-4, abs=1e-6 * np.abs(deps).max()), i


def test_invisible_anchors_and_linearity_in_the_incoming_gradients():
    prob = tiny(seed=42, N=12, C=2)
    prob["points"][0][:4, 2] += 500.0                       # behind / off the image: contribute nothing
    rng = np.random.default_rng(1)
    B = rng.normal(size=(6, 6)); GH = B + B.T; Gg = rng.normal(size=6)
    a = pb.photo_backward(prob["query_feat"][0], prob["ref_feat"][0], prob["points"][0], prob["gt_pose"], prob["K"], GH, Gg, "l2", 0.0)
    assert not np.any(a[1][:4])
    z = pb.photo_backward(prob["query_feat"][0], prob["ref_feat"][0], prob["points"][0], prob["gt_pose"], prob["K"], 0 * GH, 0 * Gg, "l2", 0.0)
    assert not np.any(z[0]) and not np.any(z[1]) and not np.any(z[2])
    b = pb.photo_backward(prob["query_feat"][0], prob["ref_feat"][0], prob["points"][0], prob["gt_pose"], prob["K"], 2 * GH, 2 * Gg, "l2", 0.0)
    assert np.allclose(b[0], 2 * a[0]) and np.allclose(b[1], 2 * a[1]) and np.allclose(b[2], 2 * a[2])

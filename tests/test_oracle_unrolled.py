"""Pins of oracle/pilot_unrolled.py (backward pass through all the LM steps of an unrolled refinement): central differences
of the FORWARD oracle's whole refinement + the per-step reprojection losses (supp Eq.7-8) with respect to single feature-map
entries, reference entries and the initial pose. CPU only."""
import numpy as np
import pytest

from oracle import pilot_oracle as po
from oracle import pilot_supervision as ps
from oracle import pilot_unrolled as pu
from tests.small_problems import tiny
from tests.test_oracle_photo_backward import _perturb

ALPHA, SCALE, ZN = 1.0, 2.0, 0.1


def two_level_problem(seed=71, N=60, C=3):
    """Two pyramid levels of the same size with different (seeded) maps and reference features, one hypothesis started off
    the ground truth."""
    a, b = tiny(seed=seed, N=N, C=C, n_hyp=1), tiny(seed=seed + 1, N=N, C=C, n_hyp=1)
    p = dict(a)
    p["n_levels"] = 2
    for k in ("width", "height", "channels", "query_feat", "query_conf", "intrinsics", "points", "ref_feat"):
        p[k] = [a[k][0], b[k][0] if k in ("query_feat", "ref_feat") else a[k][0]]
    p["init_poses"] = _perturb(a["gt_pose"], np.array([0.9, -0.6, 0.5, 0.012, -0.01, 0.008])).astype(np.float32)[None]
    return p


def fd_entry(prob, params, key, l, idx):
    """Median of three central differences (widths 2^-9 .. 2^-11) of the total loss with respect to one entry of level l's
    map or reference features: the refinement is only piecewise smooth (bilinear cells, accept / reject), one width may
    straddle a jump."""
    a0 = prob[key][l]
    est = []
    for h in (2.0 ** -9, 2.0 ** -10, 2.0 ** -11):
        vals = []
        for sgn in (+1, -1):
            ap = a0.copy(); ap[idx] = np.float32(a0[idx] + sgn * h)
            p2 = dict(prob); p2[key] = list(prob[key]); p2[key][l] = ap
            vals.append(total_loss(p2, params)[0])
        est.append((vals[0] - vals[1]) / (float(np.float32(a0[idx] + h)) - float(np.float32(a0[idx] - h))))
    return float(np.median(est))


def total_loss(prob, params, w=None):
    o = po.run(po.Bound(prob, params))
    T = sum(params["iters"])
    poses = np.concatenate([o["iter_poses"][1:, 0], o["poses64"][:1]])
    Lr = ps.reprojection_loss(poses, np.asarray(prob["gt_pose"], np.float32), prob["points"][0], [float(np.float32(k)) for k in prob["intrinsics"][0]],
                              prob["width"][0], prob["height"][0], ZN, ALPHA, SCALE)[0]
    w = np.full(T, 1.0 / T) if w is None else np.asarray(w)
    return float(np.sum(w * Lr)), o


@pytest.mark.parametrize("params", [
    dict(iters=[2, 2], loss="l2", loss_scale=0.0, lm_mode="fixed", lambda_init=3.0),
    dict(iters=[1, 3], loss="huber", loss_scale=0.4, lm_mode="adaptive", lambda_init=0.5, damp_mode="diag"),
    dict(iters=[3, 1], loss="cauchy", loss_scale=0.5, lm_mode="adaptive", lambda_init=1e-4),
])
def test_chain_matches_central_differences_of_the_forward_oracle(params):
    params = dict(params, min_valid=4, w_gravity=0.0, range_mode="off", z_near=ZN)
    prob = two_level_problem()
    L0, o0 = total_loss(prob, params)
    K32 = [float(np.float32(k)) for k in prob["intrinsics"][0]]
    g = pu.unrolled_backward(prob, params, o0, np.asarray(prob["gt_pose"], np.float32), prob["points"][0], K32,
                             prob["width"][0], prob["height"][0], ALPHA, SCALE)
    assert g["loss"][0] == pytest.approx(L0, rel=1e-12)
    for l in range(2):
        gF, gR = g["grad_feat"][l], g["grad_ref"][l]
        idx = np.argwhere(np.abs(gF) > 0.25 * np.abs(gF).max())[:4]
        assert len(idx) >= 2
        for y, x, c in idx:
            assert fd_entry(prob, params, "query_feat", l, (y, x, c)) == pytest.approx(gF[y, x, c], rel=1e-3, abs=1e-4 * np.abs(gF).max()), (l, y, x, c)
        for j, c in np.argwhere(np.abs(gR) > 0.25 * np.abs(gR).max())[:3]:
            assert fd_entry(prob, params, "ref_feat", l, (j, c)) == pytest.approx(gR[j, c], rel=1e-3, abs=1e-4 * np.abs(gR).max()), (l, j, c)
    # the initial pose: left perturbation of T_cw along each of the six directions. The refinement is only PIECEWISE smooth in
    # the pose (an anchor that crosses into the next bilinear cell changes gx, gy and with them every later step), so the
    # derivative is compared with the median of three central differences of different widths: one may straddle a jump.
    for d in range(6):
        est = []
        for he in ((1e-4, 3e-4, 1e-3) if d < 3 else (1e-5, 3e-5, 1e-4)):
            e = np.zeros(6); e[d] = he
            vals = []
            for sgn in (+1, -1):
                p2 = dict(prob)
                p2["init_poses"] = _perturb(prob["init_poses"][0].astype(np.float64), sgn * e)[None].astype(np.float32)
                vals.append(total_loss(p2, params)[0])
            est.append((vals[0] - vals[1]) / (2 * he))
        assert float(np.median(est)) == pytest.approx(g["grad_init_pose"][0, d], rel=5e-2, abs=5e-3 * np.abs(g["grad_init_pose"]).max()), (d, est)


def stuck_problem():
    """A rough (unsmoothed) map with few anchors on which the adaptive rule rejects two solves in the middle of the run
    (found by search over seeds): accepted, accepted, rejected, rejected, accepted, accepted - across the change of level."""
    a = tiny(seed=99, N=10, C=4, n_hyp=1, smooth=False)
    prob = dict(a)
    prob["n_levels"] = 2
    for k in ("width", "height", "channels", "query_feat", "query_conf", "intrinsics", "points", "ref_feat"):
        prob[k] = [a[k][0], a[k][0]]
    params = dict(iters=[4, 2], loss="cauchy", loss_scale=0.3, lm_mode="adaptive", lambda_init=1e-3, min_valid=4, w_gravity=0.0,
                  range_mode="off", z_near=ZN)
    prob["init_poses"] = _perturb(prob["gt_pose"], np.array([3.0, -2.5, 2.0, 0.05, -0.04, 0.05])).astype(np.float32)[None]
    return prob, params


def test_rejected_steps_pass_the_gradient_through():
    """The chain must pass dL/d eps through the rejected solves, still count the supervision of the repeated pose, and pick
    the chain up again at the accepted solves that follow."""
    prob, params = stuck_problem()
    L0, o0 = total_loss(prob, params)
    poses = np.concatenate([o0["iter_poses"][:, 0], o0["poses64"][:1]])
    rejected = [bool(np.array_equal(poses[r + 1], poses[r])) for r in range(6)]
    assert rejected == [False, False, True, True, False, False]
    K32 = [float(np.float32(k)) for k in prob["intrinsics"][0]]
    g = pu.unrolled_backward(prob, params, o0, np.asarray(prob["gt_pose"], np.float32), prob["points"][0], K32,
                             prob["width"][0], prob["height"][0], ALPHA, SCALE)
    assert g["loss"][0] == pytest.approx(L0, rel=1e-12)
    gR, gF = g["grad_ref"][0], g["grad_feat"][0]
    for j, c in np.argwhere(np.abs(gR) > 0.25 * np.abs(gR).max())[:3]:
        assert fd_entry(prob, params, "ref_feat", 0, (j, c)) == pytest.approx(gR[j, c], rel=1e-3, abs=1e-4 * np.abs(gR).max()), (j, c)
    for y, x, c in np.argwhere(np.abs(gF) > 0.25 * np.abs(gF).max())[:3]:
        assert fd_entry(prob, params, "query_feat", 0, (y, x, c)) == pytest.approx(gF[y, x, c], rel=1e-3, abs=1e-4 * np.abs(gF).max()), (y, x, c)

"""CPU ORACLE of the backward pass through ALL the LM steps of an unrolled refinement, numpy float64.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import this
module. It shares no code with paper_2606_31098_b200/csrc.

What it is (supp III-C): "Training is performed by unrolling the feature-metric pose
refinement process ... the final supervision is applied on the geometric reprojection error after each refinement step ...
the refinement is unrolled over nine coarse-to-fine steps, and the final training objective averages the reprojection losses
over all unrolled steps." With T^r the pose after r solves (T^0 the initial pose, T = sum(iters) solves over the levels) and
    L = sum_{r=1..T} w_r L_r(T^r)          (L_r: supp Eq.8, pilot_supervision.reprojection_loss; the paper: w_r = 1/T)
the forward chain is, per solve r at level l(r) (SURVEY.md 8(c) algorithm):
    (H_r, g_r) = photo term at T^r on level l(r);   dxi_r = -(H_r + lambda_r D)^-1 g_r  (Eq.8);
    accepted:  T^{r+1} = exp(dxi_r^) T^r  (Eq.9);    rejected / factorisation failed:  T^{r+1} = T^r.
The chain rule, read from the last pose backwards with q = dL/d eps at the current pose (eps the left perturbation of T_cw,
readings A1, A2, A25 of DESIGN.md), composes the three pinned pieces - nothing else:
    q_T = w_T dL_T/d eps                                              (pilot_supervision.reprojection_loss_grad)
    for r = T-1 .. 0:
        accepted:  (dxi, G_H, G_g, q_pass) = lm_step_adjoint(H_r, g_r, lambda_r, q)      (pilot_supervision)
                   (dF, dref, deps, dconf)  = photo_backward(level l(r), T^r, G_H, G_g)  (pilot_photo_backward); accumulate
                   q = q_pass + deps
        rejected:  q stays
        if r >= 1: q += w_r dL_r/d eps
lambda_r and the accept / reject decisions are piecewise constant in the inputs and held fixed (as are visible sets and
bilinear cells). Whether solve r was accepted is read off the forward oracle's iterates: the pose changed.
Pins (tests/test_oracle_unrolled.py): central differences of the FORWARD oracle's whole multi-step, multi-level refinement
followed by the loss, with respect to single map entries, reference entries and the initial pose.
"""
import numpy as np

from oracle import pilot_photo_backward as pb
from oracle import pilot_supervision as ps


def _decode(a, dtype):
    a = np.asarray(a)
    if dtype == "bf16":
        return (a.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    return a.astype(np.float64)


def unrolled_backward(prob, params, orc, pose_star, sup_points, sup_K, width, height, alpha, scale, step_weights=None):
    """prob: problem dict (workloads / small_problems); params: the parameter dict the forward oracle ran with (priors off);
    orc: what pilot_oracle.run returned for them. Returns dict(grad_feat [L] of [Hh][W][C], grad_ref [L] of [N][C],
    grad_conf [L] of [Hh][W] or None, grad_init_pose [H][6], loss [H])."""
    iters = list(params["iters"])
    L, T, H = len(iters), int(sum(iters)), orc["poses64"].shape[0]
    z_near = float(params.get("z_near", 0.1))
    loss, loss_scale = params.get("loss", "huber"), float(params.get("loss_scale", 0.1))
    damp_diag = params.get("damp_mode", "identity") == "diag"
    w = np.full(max(T, 1), 1.0 / max(T, 1)) if step_weights is None else np.asarray(step_weights, np.float64)
    level_of = [l for l in range(L) for _ in range(iters[l])]
    feat = [_decode(prob["query_feat"][l], prob["dtype"]) for l in range(L)]
    ref = [_decode(prob["ref_feat"][l], prob["dtype"]) for l in range(L)]
    confs = prob.get("query_conf", [None] * L)
    out = dict(grad_feat=[np.zeros_like(f) for f in feat], grad_ref=[np.zeros_like(r) for r in ref],
               grad_conf=[None if c is None else np.zeros(np.asarray(c).shape) for c in confs],
               grad_init_pose=np.zeros((H, 6)), loss=np.zeros(H))
    for m in range(H):
        poses = [orc["iter_poses"][r, m] for r in range(T)] + [orc["poses64"][m]]          # T^0 .. T^T
        if T == 0:
            continue
        Lr, _, dLr = ps.reprojection_loss_grad(np.stack(poses[1:]), pose_star, sup_points, sup_K, width, height, z_near, alpha, scale)
        out["loss"][m] = float(np.sum(w[:T] * Lr))
        q = w[T - 1] * dLr[T - 1]
        for r in range(T - 1, -1, -1):
            l = level_of[r]
            if not np.array_equal(poses[r + 1], poses[r]):                                  # accepted
                _, GH, Gg, q_pass = ps.lm_step_adjoint(orc["iter_hessian"][r, m].astype(np.float64).reshape(6, 6),
                                                       orc["iter_gradient"][r, m].astype(np.float64),
                                                       float(orc["iter_lambda"][r, m]), damp_diag, q)
                dF, dref, deps, _, dconf = pb.photo_backward(feat[l], ref[l], prob["points"][l], poses[r], prob["intrinsics"][l],
                                                             GH, Gg, loss, loss_scale, z_near, confs[l])
                out["grad_feat"][l] += dF
                out["grad_ref"][l] += dref
                if dconf is not None:
                    out["grad_conf"][l] += dconf
                q = q_pass + deps
            if r >= 1:
                q = q + w[r - 1] * dLr[r - 1]
        out["grad_init_pose"][m] = q
    return out

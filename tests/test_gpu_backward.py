"""pilot_refine_photo_backward against oracle/pilot_photo_backward.py (pinned by central differences of the forward oracle),
and the chain rule through one whole unrolled LM step (loss gradient -> step adjoint -> photo backward) against central
differences of the forward ORACLE's one-step refinement."""
import numpy as np
import pytest

from oracle import pilot_photo_backward as pb
from tests.small_problems import tiny

pytestmark = pytest.mark.gpu


def _decode(prob, a):
    import torch
    if prob["dtype"] == "f32":
        return np.asarray(a, np.float64)
    dt = torch.bfloat16 if prob["dtype"] == "bf16" else torch.float16
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).view(dt).double().numpy().reshape(np.shape(a))


@pytest.mark.parametrize("dtype,C,loss,scale,conf", [("f32", 3, "huber", 0.25, True), ("f32", 16, "l2", 0.0, False),
                                                     ("bf16", 32, "cauchy", 0.3, True), ("f16", 64, "huber", 0.2, False),
                                                     ("bf16", 40, "cauchy", 0.5, False)])
def test_photo_backward_matches_the_oracle(dtype, C, loss, scale, conf):
    import torch
    from paper_2606_31098_b200 import binding
    prob = tiny(seed=50 + C, N=200, C=C, n_hyp=3, dtype=dtype, conf=conf)
    rng = np.random.default_rng(C)
    n = 3
    GH = rng.normal(size=(n, 6, 6)); GH = (GH + GH.transpose(0, 2, 1)).astype(np.float32)
    Gg = rng.normal(size=(n, 6)).astype(np.float32)
    di = binding.DeviceInputs(prob)
    d = torch.device("cuda")
    out = binding.photo_backward(di, 0, torch.from_numpy(prob["init_poses"]).to(d), torch.from_numpy(GH.reshape(n, 36)).to(d),
                                 torch.from_numpy(Gg).to(d), loss, scale, 0.1)
    torch.cuda.synchronize()
    F, ref = _decode(prob, prob["query_feat"][0]), _decode(prob, prob["ref_feat"][0])
    K32 = [float(np.float32(k)) for k in prob["K"]]
    qc = prob["query_conf"][0] if conf else None
    dF, dref, dconf, dpose = 0.0, 0.0, 0.0, []
    for m in range(n):
        o = pb.photo_backward(F, ref, prob["points"][0], prob["init_poses"][m], K32, GH[m], Gg[m], loss, float(np.float32(scale)),
                              float(np.float32(0.1)), qc)
        dF, dref = dF + o[0], dref + o[1]
        dpose.append(o[2])
        if conf:
            dconf = dconf + o[4]
    tol = 2e-4          # fp32 per-channel arithmetic and fp32 atomic sums on the GPU
    g = out["grad_feat"].cpu().numpy()
    assert np.abs(g - dF).max() <= tol * np.abs(dF).max()
    assert np.abs(out["grad_ref"].cpu().numpy() - dref).max() <= tol * np.abs(dref).max()
    dp = np.array(dpose)
    assert np.abs(out["grad_pose"].cpu().numpy() - dp).max() <= tol * np.abs(dp).max()
    if conf:
        assert np.abs(out["grad_conf"].cpu().numpy() - dconf).max() <= tol * np.abs(dconf).max()
    else:
        assert out["grad_conf"] is None


def test_chain_rule_through_one_unrolled_lm_step():
    """L(F) = reprojection loss of the pose after ONE LM step (photo term only, L2 loss, fixed lambda). GPU: loss gradient
    at the updated pose -> lm_step_adjoint on the recorded system -> photo_backward at the initial pose. Expected: central
    differences of the forward ORACLE's one-step run with respect to single map and reference entries."""
    import torch
    from oracle import pilot_oracle as po
    from oracle import pilot_supervision as ps
    from paper_2606_31098_b200 import binding
    prob = tiny(seed=61, N=120, C=4, n_hyp=1)
    params = dict(iters=[1], loss="l2", loss_scale=0.0, lm_mode="fixed", lambda_init=5.0, min_valid=4, w_gravity=0.0, range_mode="off")
    pts, K, W, H = prob["points"][0], prob["intrinsics"][0], prob["width"][0], prob["height"][0]
    K32 = [float(np.float32(k)) for k in K]
    Tstar = np.asarray(prob["gt_pose"], np.float32)
    # start off the ground truth so that the loss has a gradient
    from tests.test_oracle_photo_backward import _perturb
    prob["init_poses"][0] = _perturb(prob["gt_pose"], np.array([0.8, -0.5, 0.6, 0.01, -0.008, 0.012])).astype(np.float32)

    def loss_of(p):
        o = po.run(po.Bound(p, params))
        return ps.reprojection_loss(o["poses64"][:1], Tstar, pts, K32, W, H, 0.1, 1.0, 2.0)[0][0], o

    L0, o0 = loss_of(prob)
    d = torch.device("cuda")
    di = binding.DeviceInputs(prob)
    gpu = binding.refine(prob, params)
    T1 = torch.from_numpy(gpu["poses"][:1]).to(d)
    _, _, q = binding.reprojection_loss_grad(T1, Tstar, torch.from_numpy(pts).to(d), K, W, H, 0.1, 1.0, 2.0)
    adj = binding.lm_step_adjoint(torch.from_numpy(gpu["iter_hessian"][0]).to(d), torch.from_numpy(gpu["iter_gradient"][0]).to(d),
                                  torch.from_numpy(gpu["iter_lambda"][0]).to(d), q, "identity")
    bw = binding.photo_backward(di, 0, torch.from_numpy(prob["init_poses"]).to(d), adj["grad_hessian"], adj["grad_gradient"], "l2", 0.0, 0.1)
    torch.cuda.synchronize()
    gF, gR = bw["grad_feat"].cpu().numpy(), bw["grad_ref"].cpu().numpy()
    F0, r0 = prob["query_feat"][0], prob["ref_feat"][0]
    h = 2.0 ** -6
    idx = np.argwhere(np.abs(gF) > 0.2 * np.abs(gF).max())[:6]
    assert len(idx) >= 3
    for y, x, c in idx:
        vals = []
        for sgn in (+1, -1):
            Fp = F0.copy(); Fp[y, x, c] = np.float32(F0[y, x, c] + sgn * h)
            p2 = dict(prob); p2["query_feat"] = [Fp]
            vals.append(loss_of(p2)[0])
        step = float(np.float32(F0[y, x, c] + h)) - float(np.float32(F0[y, x, c] - h))
        assert (vals[0] - vals[1]) / step == pytest.approx(gF[y, x, c], rel=2e-2, abs=2e-3 * np.abs(gF).max()), (y, x, c)
    jdx = np.argwhere(np.abs(gR) > 0.2 * np.abs(gR).max())[:4]
    for j, c in jdx:
        vals = []
        for sgn in (+1, -1):
            rp = r0.copy(); rp[j, c] = np.float32(r0[j, c] + sgn * h)
            p2 = dict(prob); p2["ref_feat"] = [rp]
            vals.append(loss_of(p2)[0])
        step = float(np.float32(r0[j, c] + h)) - float(np.float32(r0[j, c] - h))
        assert (vals[0] - vals[1]) / step == pytest.approx(gR[j, c], rel=2e-2, abs=2e-3 * np.abs(gR).max()), (j, c)

"""pilot_refine_unrolled_backward (the backward pass through every LM step of an unrolled refinement, SURVEY.md 8(f).4,
supp III-C PAPER.md:427-440) against oracle/pilot_unrolled.py, which is pinned by central differences of the forward oracle
(tests/test_oracle_unrolled.py). Each side differentiates ITS OWN forward run of the same inputs."""
import numpy as np
import pytest

from tests.small_problems import tiny
from tests.test_oracle_photo_backward import _perturb
from tests.test_oracle_unrolled import stuck_problem, two_level_problem

pytestmark = pytest.mark.gpu

ALPHA, SCALE, ZN = 1.0, 2.0, 0.1


def with_hypotheses(prob, n, seed=5):
    rng = np.random.default_rng(seed)
    poses = [_perturb(prob["gt_pose"], np.concatenate([rng.uniform(-1, 1, 3), rng.uniform(-0.015, 0.015, 3)])) for _ in range(n)]
    p = dict(prob)
    p["init_poses"] = np.stack(poses).astype(np.float32)
    return p


def gpu_and_oracle(prob, params, mode="auto", weights=None, teacher=False, sup_level=0):
    """GPU forward with the extra records + GPU chain, oracle forward + oracle chain. teacher=True: the GPU chain reads the
    ORACLE's records (rounded to fp32 and uploaded) instead of its own forward's, so that both chains differentiate the very
    same trajectory - for inputs whose free-running trajectories drift apart (rough maps, bf16 features)."""
    import torch
    from oracle import pilot_oracle as po
    from oracle import pilot_unrolled as pu
    from paper_2606_31098_b200 import binding
    d = torch.device("cuda")
    di = binding.DeviceInputs(prob)
    r = binding.Refiner.for_inputs(di, params)
    r.set_exec_mode(mode, 0)
    r.record_iterates(True)
    out = r.run(di, params)
    torch.cuda.synchronize()
    out_np = {k: v.cpu().numpy().copy() for k, v in out.items()}
    sl = sup_level                          # the level whose camera and anchors define the reprojection supervision
    pts = torch.from_numpy(np.ascontiguousarray(prob["points"][sl], np.float32)).to(d)
    K = prob["intrinsics"][sl]
    Tstar = np.asarray(prob["gt_pose"], np.float32)
    orc = po.run(po.Bound(prob, params))
    T, H = orc["iter_poses"].shape[:2]
    nxt = np.concatenate([orc["iter_poses"][1:], orc["poses64"][None]])
    acc = np.array([[not np.array_equal(nxt[t, m], orc["iter_poses"][t, m]) for m in range(H)] for t in range(T)])
    rec = out
    if teacher:
        up = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dt)).to(d)
        rec = dict(iter_hessian=up(orc["iter_hessian"], np.float32), iter_gradient=up(orc["iter_gradient"], np.float32),
                   iter_lambda=up(orc["iter_lambda"], np.float32), iter_poses=up(orc["iter_poses"], np.float32),
                   iter_accept=up(acc, np.int32), poses=up(orc["poses64"], np.float32))
    g = binding.unrolled_backward(r, di, params, rec, Tstar, pts, K, prob["width"][sl], prob["height"][sl], ALPHA, SCALE,
                                  step_weights=weights, grad_conf=True)
    torch.cuda.synchronize()
    K32 = [float(np.float32(k)) for k in K]
    og = pu.unrolled_backward(prob, params, orc, Tstar, prob["points"][sl], K32, prob["width"][sl], prob["height"][sl], ALPHA, SCALE,
                              step_weights=weights)
    r.close()
    return dict(out=out_np, g=g, orc=orc, og=og, acc=acc, first_level_solves=int(params["iters"][0]))


def check(res, n_levels, tol, pose_tol=1e-3, strict_accept=True):
    """pose_tol: the free-running iterates against the oracle's (north_star: 1e-3 for fp32 features, 5e-3 for bf16).
    strict_accept=False: near convergence the cost differences that decide accept / reject are at the level of the bf16
    rounding, so the free-running GPU run may reject a late step the oracle accepts (reading A19: compare what is unique) -
    the flags must then agree on every solve of the first level and on at least 80 % of all solves."""
    out, g, og = res["out"], res["g"], res["og"]
    # the extra records of the forward run: iterate poses and accept flags
    assert np.abs(out["iter_poses"] - res["orc"]["iter_poses"]).max() <= pose_tol
    if strict_accept:
        assert np.array_equal(out["iter_accept"].astype(bool), res["acc"])
    else:
        same = out["iter_accept"].astype(bool) == res["acc"]
        assert same[:res["first_level_solves"]].all() and same.mean() >= 0.8, same
    assert np.allclose(g["loss"].cpu().numpy(), og["loss"], rtol=tol, atol=1e-6)
    gi = g["grad_init_pose"].cpu().numpy()
    assert np.abs(gi - og["grad_init_pose"]).max() <= tol * np.abs(og["grad_init_pose"]).max()
    for l in range(n_levels):
        for key in ("grad_feat", "grad_ref", "grad_conf"):
            if og[key][l] is None:
                continue
            a, b = g[key][l].cpu().numpy(), og[key][l]
            assert np.abs(a - b).max() <= tol * max(np.abs(b).max(), 1e-30), (l, key, np.abs(a - b).max(), np.abs(b).max())


@pytest.mark.parametrize("mode", ["passes", "split", "resident"])
@pytest.mark.parametrize("params", [
    dict(iters=[2, 2], loss="l2", loss_scale=0.0, lm_mode="fixed", lambda_init=3.0),
    dict(iters=[1, 3], loss="huber", loss_scale=0.4, lm_mode="adaptive", lambda_init=0.5, damp_mode="diag"),
    dict(iters=[3, 1], loss="cauchy", loss_scale=0.5, lm_mode="adaptive", lambda_init=1e-4),
])
def test_chain_matches_the_oracle(params, mode):
    params = dict(params, min_valid=4, w_gravity=0.0, range_mode="off", z_near=ZN)
    prob = with_hypotheses(two_level_problem(C=4), 3)
    check(gpu_and_oracle(prob, params, mode), 2, 2e-3)


def test_confidence_maps_weights_and_bf16():
    """Query confidence maps (their gradient too), non-uniform step weights, and bf16 features (the forward runs on the
    tensor-core path where it applies; the backward reads the same bf16 maps)."""
    a, b = tiny(seed=81, N=80, C=32, n_hyp=1, conf=True, dtype="bf16", W=48, H=36), tiny(seed=82, N=80, C=32, n_hyp=1, conf=True, dtype="bf16", W=48, H=36)
    p = dict(a)
    p["n_levels"] = 2
    for k in ("width", "height", "channels", "query_feat", "query_conf", "intrinsics", "points", "ref_feat"):
        p[k] = [a[k][0], b[k][0] if k in ("query_feat", "ref_feat", "query_conf") else a[k][0]]
    p = with_hypotheses(p, 2, seed=9)
    params = dict(iters=[2, 2], loss="huber", loss_scale=0.5, lm_mode="adaptive", lambda_init=1.0, min_valid=4, w_gravity=0.0,
                  range_mode="off", z_near=ZN)
    check(gpu_and_oracle(p, params, "auto", weights=[0.1, 0.2, 0.3, 0.4], teacher=True), 2, 2e-3, pose_tol=5e-3)


def test_paper_shape_nine_unrolled_steps():
    """The paper's own training shape (supp III-B/C): 500 geo-anchors, a three-level pyramid of L2-normalised
    32-channel descriptors with query and reference confidences, 2 + 3 + 4 = nine unrolled steps, the objective the average
    of the nine per-step reprojection losses in the full-resolution camera. Synthetic stand-in for its data
    (workloads.paper_frame); priors off (the chain differentiates the photo term)."""
    from paper_2606_31098_b200 import workloads as wl
    prob = wl.paper_frame(N=500, iters=(2, 3, 4), dtype="bf16")
    params = dict(prob["params"], w_gravity=0.0, range_mode="off")
    rng = np.random.default_rng(17)
    prob["init_poses"] = np.stack([_perturb(prob["gt_pose"], np.concatenate([rng.uniform(-3, 3, 3), rng.uniform(-0.02, 0.02, 3)]))
                                   for _ in range(2)]).astype(np.float32)
    res = gpu_and_oracle(prob, params, "auto", teacher=True, sup_level=2)
    assert res["out"]["iter_accept"].shape == (9, 2) and res["out"]["iter_accept"].sum() >= 12
    check(res, 3, 2e-3, pose_tol=5e-3, strict_accept=False)
    assert float(res["g"]["loss"].min()) > 0.0


def test_rejected_steps():
    prob, params = stuck_problem()
    res = gpu_and_oracle(prob, params, "passes", teacher=True)
    assert res["out"]["iter_accept"][:, 0].tolist() == [1, 1, 0, 0, 1, 1]
    check(res, 2, 2e-3, pose_tol=5e-3)         # ten anchors on a rough map: the free-running iterates drift by millimetres


def test_argument_errors():
    import ctypes as C
    import torch
    from paper_2606_31098_b200 import binding
    prob = with_hypotheses(two_level_problem(C=4), 2)
    params = dict(iters=[1, 1], loss="l2", lm_mode="fixed", lambda_init=1.0, min_valid=4, w_gravity=0.0, range_mode="off", z_near=ZN)
    di = binding.DeviceInputs(prob)
    r = binding.Refiner.for_inputs(di, params)
    r.record_iterates(True)
    out = r.run(di, params)
    pts = torch.from_numpy(np.ascontiguousarray(prob["points"][0], np.float32)).cuda()
    args = (np.asarray(prob["gt_pose"], np.float32), pts, prob["intrinsics"][0], prob["width"][0], prob["height"][0], ALPHA, SCALE)
    with pytest.raises(RuntimeError, match="-3"):                       # priors on: not part of this chain
        binding.unrolled_backward(r, di, dict(params, w_gravity=1.0), out, *args)
    with pytest.raises(RuntimeError, match="-3"):
        binding.unrolled_backward(r, di, dict(params, grad_mode="central_sampled"), out, *args)
    assert binding.lib().pilot_refine_unrolled_backward_scratch_bytes(2, 2) > 0
    assert binding.lib().pilot_refine_unrolled_backward_scratch_bytes(-1, 2) == 0
    par, _ = binding.make_params(params, 2)
    rec, sup, g = binding.UnrolledRecords(), binding.Supervision(), binding.UnrolledGrads()
    rc = binding.lib().pilot_refine_unrolled_backward(C.byref(r.cfg), C.byref(di.inp), C.byref(par), C.byref(rec), C.byref(sup), C.byref(g),
                                                      None, 0, None)
    assert rc == -1                                                      # NULL records
    r.close()

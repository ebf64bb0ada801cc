"""pilot_refine_run_static (include/pilot_refine.h): the refinement with the library's file-scope workspace, for callers
that may not allocate. Checked against the handle path (pilot_refine_create + pilot_refine_run) on the same inputs, on two
calls in a row whose inputs differ (the shared workspace keeps the first call's contents), within the tolerances of
tests/test_gpu_parity.py. Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = {"f32": (1e-4, 1e-3), "bf16": (5e-3, 5e-3)}      # (H, g, cost relative; pose rad / m), as tests/test_gpu_parity.py
NAMES = ("poses", "cost", "n_valid", "status", "iter_hessian", "iter_gradient", "iter_cost", "iter_lambda")


def _out_tensors(torch, H, T):
    dev = torch.device("cuda", 0)
    f = lambda *s: torch.full(s, float("nan"), dtype=torch.float32, device=dev)   # noqa: E731
    return dict(poses=f(H, 12), cost=f(H), n_valid=torch.full((H,), -7, dtype=torch.int32, device=dev),
                status=torch.full((H,), -7, dtype=torch.int32, device=dev), iter_hessian=f(T, H, 36),
                iter_gradient=f(T, H, 6), iter_cost=f(T, H), iter_lambda=f(T, H))


def _handle_path(binding, torch, di, P):
    r = binding.Refiner.for_inputs(di, P)
    out = r.run(di, P)
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy().copy() for k, v in out.items()}
    plan = r.last_plan()
    launches = r.last_launches
    r.close()
    return res, launches, plan


def _compare(got, want, dtype):
    from tests import parity
    tol_sys, tol_pose = TOL[dtype]
    assert np.array_equal(got["n_valid"], want["n_valid"])
    assert np.array_equal(got["status"], want["status"])
    for rec in range(want["iter_cost"].shape[0]):
        Hg, Hw = got["iter_hessian"][rec].astype(np.float64), want["iter_hessian"][rec].astype(np.float64)
        gg, gw = got["iter_gradient"][rec].astype(np.float64), want["iter_gradient"][rec].astype(np.float64)
        assert (np.linalg.norm(Hg - Hw, axis=1) <= tol_sys * np.linalg.norm(Hw, axis=1)).all(), rec
        assert (np.linalg.norm(gg - gw, axis=1) <= tol_sys * np.maximum(np.linalg.norm(gw, axis=1), 1e-30)).all(), rec
        assert np.allclose(got["iter_cost"][rec], want["iter_cost"][rec], rtol=tol_sys, atol=0, equal_nan=True), rec
        assert np.allclose(got["iter_lambda"][rec], want["iter_lambda"][rec], rtol=1e-6, atol=0), rec
    assert np.allclose(got["cost"], want["cost"], rtol=tol_sys, atol=0, equal_nan=True)
    assert parity.rot_angle(got["poses"], want["poses"]).max() <= tol_pose
    assert parity.trans_dist(got["poses"], want["poses"]).max() <= tol_pose


def _problems(kind):
    from paper_2606_31098_b200 import workloads as wl
    if kind == "resident":      # small levels: the cluster-resident kernel, tensor-core contraction (bf16, 32+ channels)
        return wl.config1(H=24, N=2048, iters=(3, 3, 3)), wl.config1(H=9, N=1500, iters=(3, 3, 3), idx=2), "bf16"
    # one launch per pass with ticket + last-CTA finalisation over several chunks per hypothesis
    return wl.config4(H=48, N=40000, iters=3, width=640, height=360, dsm_size=1024), \
        wl.config4(H=40, N=39000, iters=3, width=640, height=360, dsm_size=1024), "bf16"


@pytest.mark.parametrize("kind", ["resident", "passes"])
def test_static_workspace_entry_matches_the_handle_path_twice_in_a_row(kind):
    import torch
    from paper_2606_31098_b200 import binding
    first, second, dtype = _problems(kind)
    assert first["dtype"] == dtype
    cap_h = max(first["init_poses"].shape[0], second["init_poses"].shape[0])
    cap_n = max(max(len(p) for p in first["points"]), max(len(p) for p in second["points"]))
    seen_plans = []
    for prob in (first, second):             # second call: fewer hypotheses, other poses, same (dirty) workspace
        P = dict(prob.get("params", {}))
        di = binding.DeviceInputs(prob, 0)
        want, launches_want, plan = _handle_path(binding, torch, di, P)
        seen_plans.append(plan)
        H, T = di.n_hyp, sum(P["iters"])
        out = _out_tensors(torch, H, T)
        before = torch.cuda.memory_allocated(0)
        launches = binding.run_static(di, P, out, max_hypotheses=cap_h, max_points=cap_n)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated(0) == before
        assert launches == launches_want and launches > 0
        got = {k: out[k].cpu().numpy() for k in NAMES}
        _compare(got, want, dtype)
    if kind == "resident":
        assert all(res != 0 for _, res in seen_plans)
    else:
        assert all(res == 0 for _, res in seen_plans)


def test_static_workspace_entry_rejects_what_does_not_fit():
    import torch
    from paper_2606_31098_b200 import binding, workloads as wl
    prob = wl.config1(H=4, N=512, iters=(1, 1, 1))
    di = binding.DeviceInputs(prob, 0)
    P = dict(prob.get("params", {}))
    out = _out_tensors(torch, 4, 3)
    limit = binding.static_workspace_bytes()
    assert limit == 32 << 20
    with pytest.raises(RuntimeError, match="workspace too small"):
        binding.run_static(di, P, out, max_hypotheses=1024, max_points=65536)      # 67 MB of partial sums
    torch.cuda.synchronize()
    assert torch.isnan(out["poses"]).all()                                         # nothing was launched
    assert binding.run_static(di, P, out, max_hypotheses=256, max_points=65536) > 0   # config 4's capacity fits
    torch.cuda.synchronize()
    assert torch.isfinite(out["poses"]).all()

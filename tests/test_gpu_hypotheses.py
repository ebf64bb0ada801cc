"""GPU-vs-oracle parity of the hypothesis-set operations (seed / select / top-k / run_levels) through the C-ABI.
Index work is bit-exact; seeded poses agree to fp32 rounding."""
import numpy as np
import pytest

from tests import parity

pytestmark = pytest.mark.gpu

PAPER_YAWS = [-9, -7, -5, -3, -1, 1, 3, 5, 7, 9]


def dev(a, dtype=None):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a if dtype is None else np.asarray(a, dtype))).cuda()


@pytest.mark.parametrize("frame", ["camera", "world"])
def test_seed_matches_oracle(frame):
    import torch
    from oracle import pilot_hypotheses as ph
    from paper_2606_31098_b200 import binding, workloads as wl
    T = wl.pitched_pose([30.0, -140.0, 160.0], 50.0, 25.0).reshape(-1).astype(np.float32)
    rng = np.random.default_rng(4)
    grid = binding.grid_offsets(10.0, 2.0, PAPER_YAWS, [0, 0, 1.0])
    assert grid.shape == (1210, 6)
    assert np.allclose(grid, ph.grid_offsets(10.0, 2.0, PAPER_YAWS, [0, 0, 1.0]), atol=1e-7)
    rnd = (rng.normal(size=(333, 6)) * [0.3, 0.3, 0.3, 20, 20, 20]).astype(np.float32)
    rnd[0] = 0
    rnd[1, :3] = [1e-9, 0, 0]                      # series branch of the rotation exponential
    for off in (grid, rnd):
        got = binding.seed_hypotheses(dev(T), dev(off), frame)
        torch.cuda.synchronize()
        want = ph.seed_hypotheses(T, off, ph.SEED_CAMERA if frame == "camera" else ph.SEED_WORLD)
        g = got.cpu().numpy().astype(np.float64).reshape(-1, 3, 4)
        w = want.reshape(-1, 3, 4)
        assert np.abs(g[:, :, :3] - w[:, :, :3]).max() <= 1.5e-7          # half an fp32 ulp at |r| <= 1 (+ margin)
        assert np.abs(g[:, :, 3] - w[:, :, 3]).max() <= 1.6e-5            # fp32 ulp at 256 m
    assert np.array_equal(binding.seed_hypotheses(dev(T), dev(rnd[:1]), frame).cpu().numpy()[0], T)
    assert binding.seed_hypotheses(dev(T), dev(np.zeros((0, 6), np.float32)), frame).shape == (0, 12)


@pytest.mark.parametrize("n", [1, 2, 33, 1024, 1210, 5000, 100000])
def test_select_best_is_exact(n):
    import torch
    from oracle import pilot_hypotheses as ph
    from paper_2606_31098_b200 import binding
    rng = np.random.default_rng(n)
    poses = rng.normal(size=(n, 12)).astype(np.float32)
    cases = [rng.normal(size=n) ** 2, np.round(rng.uniform(0, 3, n)), np.full(n, np.inf), np.full(n, np.nan)]
    c = rng.normal(size=n); c[rng.integers(0, n, max(1, n // 3))] = np.nan; c[rng.integers(0, n, max(1, n // 5))] = np.inf
    cases.append(c)
    c = np.zeros(n); c[n // 2] = -0.0
    cases.append(c)                                                       # -0.0 == +0.0: lowest index wins
    for c in cases:
        c = c.astype(np.float32)
        idx, pose, bc = binding.select_best(dev(c), dev(poses))
        torch.cuda.synchronize()
        want = ph.select_best(c)
        assert int(idx.item()) == want
        assert np.array_equal(pose.cpu().numpy(), poses[want])
        assert np.array_equal(bc.cpu().numpy(), c[want:want + 1], equal_nan=True)


@pytest.mark.parametrize("n,k", [(1, 1), (2, 1), (2, 2), (129, 128), (1000, 1000), (1210, 128), (4097, 5), (8192, 8192)])
def test_prune_topk_is_exact(n, k):
    import torch
    from oracle import pilot_hypotheses as ph
    from paper_2606_31098_b200 import binding
    rng = np.random.default_rng(1000 * n + k)
    poses = rng.normal(size=(n, 12)).astype(np.float32)
    cases = [rng.normal(size=n), np.round(rng.uniform(0, 6, n)), np.zeros(n)]
    c = rng.uniform(0, 100, n); c[rng.integers(0, n, max(1, n // 4))] = np.inf; c[rng.integers(0, n, max(1, n // 4))] = np.nan
    cases.append(c)
    for c in cases:
        c = c.astype(np.float32)
        idx, po, co = binding.prune_topk(dev(c), dev(poses), k)
        torch.cuda.synchronize()
        want = ph.prune_topk(c, k)
        assert np.array_equal(idx.cpu().numpy().astype(np.int64), want)
        assert np.array_equal(po.cpu().numpy(), poses[want])
        assert np.array_equal(co.cpu().numpy(), c[want], equal_nan=True)


def test_topk_rejects_bad_sizes():
    from paper_2606_31098_b200 import binding
    c, p = dev(np.zeros(8193, np.float32)), dev(np.zeros((8193, 12), np.float32))
    with pytest.raises(RuntimeError, match="-3"):
        binding.prune_topk(c, p, 4)
    with pytest.raises(RuntimeError, match="-1"):
        binding.prune_topk(c[:10], p[:10], 11)


@pytest.mark.parametrize("mode", ["passes", "resident"])
def test_run_levels_matches_oracle_on_level_slices(mode):
    """run_levels(b, e) == the oracle on the sub-problem made of levels [b, e); records keep the whole-run layout."""
    import torch
    from oracle import pilot_oracle as po
    from paper_2606_31098_b200 import binding, workloads as wl
    prob = wl.config1(H=24, N=1500, iters=(3, 2, 4))
    di = binding.DeviceInputs(prob)
    r = binding.Refiner.for_inputs(di, prob["params"])
    r.set_exec_mode(mode)
    for (b, e) in [(0, 1), (1, 3), (2, 3), (0, 3)]:
        for t in r.o.values():
            t.fill_(-7)
        out = r.run(di, prob["params"], levels=(b, e))
        torch.cuda.synchronize()
        gpu = {k: v.cpu().numpy() for k, v in out.items()}
        orc = po.run(po.Bound(parity.levels_slice(prob, b, e)), n_threads=8)
        base = sum(prob["params"]["iters"][:b])
        n_rec = sum(prob["params"]["iters"][b:e])
        g = dict(gpu)
        for k in ("iter_hessian", "iter_gradient", "iter_cost", "iter_lambda"):
            g[k] = gpu[k][base:base + n_rec]
            untouched = np.concatenate([gpu[k][:base].ravel(), gpu[k][base + n_rec:].ravel()])
            assert np.all(untouched == -7), k                              # levels outside the range: not written
        eH, eg, ec = parity.system_errors(g, orc, 0)
        assert max(eH.max(), eg.max(), ec.max()) <= 5e-3
        conv = parity.converged(orc)
        er, et = parity.pose_errors(g, orc)
        if conv.any():
            assert er[conv].max() <= 5e-3 and et[conv].max() <= 5e-3
        assert r.last_launches == 1 + (sum(k + 1 for k in prob["params"]["iters"][b:e]) if mode == "passes" else e - b)
    with pytest.raises(RuntimeError, match="-1"):
        r.run(di, prob["params"], levels=(2, 2))
    r.close()


def test_paper_schedule_1210_to_128():
    """supp II-C end to end: 1210 grid hypotheses -> coarse level -> top 128 -> finer levels ->
    arg-min, against the same pipeline assembled from the oracle's pieces."""
    import torch
    from oracle import pilot_hypotheses as ph
    from oracle import pilot_oracle as po
    from paper_2606_31098_b200 import binding, workloads as wl
    prob = wl.paper_frame()
    xy_range, xy_step, yaws = prob["grid"]
    up = -np.asarray(prob["gravity_world"], np.float64)
    off = binding.grid_offsets(xy_range, xy_step, yaws, up)
    assert off.shape == (1210, 6)
    di = binding.DeviceInputs(prob)
    pr = binding.PrunedRefiner(di, prob["params"], off, prob["keep"], "world")
    out = pr.run(dev(prob["prior_pose"]))
    torch.cuda.synchronize()
    g = {k: v.cpu().numpy() for k, v in out.items()}
    it = prob["params"]["iters"]
    # AUTO: 1210 hypotheses do not fit one wave of clusters -> on the coarse level one gather launch + one
    # finalisation launch per pass; the 128 kept ones run cluster-resident, one launch per level
    assert pr.launches == (1 + 2 * (it[0] + 1)) + (1 + 2) + 3
    pr.close()

    # oracle pipeline (its own seeds from the same fp32 offset table)
    seeds = ph.seed_hypotheses(prob["prior_pose"], off, ph.SEED_WORLD)
    c0 = po.run(po.Bound(parity.levels_slice(prob, 0, 1, seeds)), n_threads=16)
    keep = ph.prune_topk(c0["cost64"], prob["keep"])
    c1 = po.run(po.Bound(parity.levels_slice(prob, 1, 3, c0["poses64"][keep])), n_threads=16)
    b = ph.select_best(c1["cost64"])

    # kept set: identical except where the oracle's coarse costs tie with the 128th within the bf16 tolerance
    cut = c0["cost64"][keep[-1]]
    diff = set(g["kept_idx"].tolist()) ^ set(keep.tolist())
    assert len(diff) <= 8, len(diff)
    for m in diff:
        assert abs(c0["cost64"][m] - cut) <= 5e-3 * cut, (m, c0["cost64"][m], cut)
    # coarse objective of the kept hypotheses the two sides share
    common = [i for i, m in enumerate(g["kept_idx"]) if m in set(keep.tolist())]
    rel = np.abs(g["coarse_kept_cost"][common] - c0["cost64"][g["kept_idx"][common]]) / c0["cost64"][g["kept_idx"][common]]
    assert rel.max() <= 5e-3, (rel.max(), g["kept_idx"][common][rel > 5e-3])      # every shared kept hypothesis (measured: 1.5e-5)
    assert np.all(np.diff(g["coarse_kept_cost"]) >= 0)                      # ascending order
    # the selected pose and objective
    assert parity.rot_angle(g["best_pose"], c1["poses64"][b])[0] <= 5e-3
    assert parity.trans_dist(g["best_pose"], c1["poses64"][b])[0] <= 5e-3
    assert abs(g["best_cost"][0] - c1["cost64"][b]) <= 5e-3 * c1["cost64"][b]
    assert g["best_cost"][0] == g["cost"].min() and np.array_equal(g["best_pose"], g["poses"][int(g["best_idx"][0])])
    # and it is a localisation: the 3.1 m / -4.3 m / 2.2 deg prior error is removed
    gt = prob["gt_pose"]
    assert np.rad2deg(parity.rot_angle(g["best_pose"], gt))[0] < 0.1 and parity.trans_dist(g["best_pose"], gt)[0] < 0.3


def test_pruned_host_path_matches_the_device_path():
    """pilot_refine_submit_pruned_host (one call per frame through host buffers, two frames in flight) gives the same
    selection, bit for bit, as the five device calls of PrunedRefiner (same kernels, same order)."""
    import torch
    from paper_2606_31098_b200 import binding, workloads as wl
    prob = wl.paper_frame()
    xy_range, xy_step, yaws = prob["grid"]
    off = binding.grid_offsets(xy_range, xy_step, yaws, -np.asarray(prob["gravity_world"], np.float64))
    di = binding.DeviceInputs(prob)
    pr = binding.PrunedRefiner(di, prob["params"], off, prob["keep"], "world")
    out = pr.run(dev(prob["prior_pose"]))
    torch.cuda.synchronize()
    want_pose, want_cost = out["best_pose"].cpu().numpy(), out["best_cost"].cpu().numpy()
    want_idx = int(out["kept_idx"].cpu().numpy()[int(out["best_idx"].cpu().numpy()[0])])
    pr.close()
    hi = binding.DeviceInputs(prob, host=True)
    ph = binding.PrunedHostRefiner(hi, prob["params"], off, prob["keep"], "world")
    prior2 = prob["prior_pose"].copy(); prior2[3] += 0.7                      # a second frame with another prior, in flight too
    ph.submit(prob["prior_pose"]); ph.submit(prior2)
    r0 = {k: v.clone() for k, v in ph.wait().items()}
    ph.submit(prob["prior_pose"])
    r1 = {k: v.clone() for k, v in ph.wait().items()}
    r2 = {k: v.clone() for k, v in ph.wait().items()}
    for r in (r0, r2):
        assert np.array_equal(r["pose"].numpy(), want_pose.reshape(-1)) and r["cost"].numpy()[0] == want_cost[0]
        assert int(r["index"].numpy()[0]) == want_idx
    assert not np.array_equal(r1["pose"].numpy(), want_pose.reshape(-1))      # the other prior gave another answer
    assert parity.trans_dist(r1["pose"].numpy(), prob["gt_pose"])[0] < 0.3    # ... which is still a localisation
    with pytest.raises(RuntimeError):
        ph.submit(prob["prior_pose"]); ph.submit(prob["prior_pose"]); ph.submit(prob["prior_pose"])   # third in flight
    ph.wait(); ph.wait()
    ph.close()

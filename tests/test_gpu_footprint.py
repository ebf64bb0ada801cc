"""GPU-vs-oracle parity of the reference-crop geometry (supp Eq.2-3) through the C-ABI."""
import numpy as np
import pytest

from tests import parity

pytestmark = pytest.mark.gpu


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, np.float32)).cuda()


def scene():
    from paper_2606_31098_b200 import workloads as wl
    prob = wl.config1(H=16, N=2048, iters=(3, 3, 3))
    K = prob["intrinsics"][2]
    return prob, K, 480, 270


@pytest.mark.parametrize("n_samples", [1, 31, 64, 1000, 4097])
def test_footprint_matches_oracle(n_samples):
    import torch
    from oracle import pilot_footprint as pf
    from paper_2606_31098_b200 import binding
    prob, K, W, H = scene()
    pose32 = prob["gt_pose"].astype(np.float32)
    s_max = 900.0
    got = binding.footprint(dev(pose32), K, W, H, dev(prob["dsm"]), prob["dsm_origin"], prob["dsm_gsd"], n_samples, s_max)
    torch.cuda.synchronize()
    got = got.cpu().numpy().astype(np.float64)
    Kf = [float(np.float32(k)) for k in K]
    want = pf.footprint(pose32.astype(np.float64), Kf, W, H, prob["dsm"], prob["dsm_origin"], prob["dsm_gsd"], n_samples, s_max)
    C = pose32.reshape(3, 4)[:, 3].astype(np.float64)
    for c in range(4):
        if np.isnan(want[c, 0]):
            assert np.all(np.isnan(got[c]))
            continue
        # the same sample index on both sides (the arg-min is an integer decision taken in double on both)
        ig = np.linalg.norm(got[c, :3] - C) / (s_max / n_samples)
        iw = np.linalg.norm(want[c, :3] - C) / (s_max / n_samples)
        assert round(ig) == round(iw), (c, ig, iw)
        assert np.abs(got[c, :3] - want[c, :3]).max() <= 6.2e-5          # fp32 ulp at 512-1024 m
        assert abs(got[c, 3] - want[c, 3]) <= 1e-4 + 1e-6 * want[c, 3]


def test_footprint_off_the_map_is_nan_and_argument_errors():
    import torch
    from paper_2606_31098_b200 import binding, workloads as wl
    prob, K, W, H = scene()
    far = wl.pitched_pose([5000.0, 5000.0, 100.0], 45.0).reshape(-1)
    got = binding.footprint(dev(far), K, W, H, dev(prob["dsm"]), prob["dsm_origin"], prob["dsm_gsd"], 100, 300.0)
    torch.cuda.synchronize()
    assert np.all(np.isnan(got.cpu().numpy()))
    with pytest.raises(RuntimeError, match="-1"):
        binding.footprint(dev(far), K, W, H, dev(prob["dsm"]), prob["dsm_origin"], prob["dsm_gsd"], 0, 300.0)


def test_lift_anchors_matches_oracle_and_feeds_the_refinement():
    import torch
    from oracle import pilot_footprint as pf
    from oracle import pilot_oracle as po
    from paper_2606_31098_b200 import binding, workloads as wl
    prob, K, W, H = scene()
    pose32 = prob["gt_pose"].astype(np.float32)
    dsm_d = dev(prob["dsm"])
    corners = binding.footprint(dev(pose32), K, W, H, dsm_d, prob["dsm_origin"], prob["dsm_gsd"], 2000, 900.0)
    rng = np.random.default_rng(8)
    Wc = Hc = 512                                                 # "resized to 512"
    pix = rng.uniform([0, 0], [Wc - 1, Hc - 1], (2048 + 13, 2)).astype(np.float32)
    pix[:4] = [[0, 0], [Wc - 1, 0], [Wc - 1, Hc - 1], [0, Hc - 1]]
    pts = binding.lift_anchors(corners, Wc, Hc, dev(pix), dsm_d, prob["dsm_origin"], prob["dsm_gsd"])
    torch.cuda.synchronize()
    c_np, got = corners.cpu().numpy(), pts.cpu().numpy()
    want = pf.lift_anchors(c_np.astype(np.float64), Wc, Hc, pix.astype(np.float64), prob["dsm"], prob["dsm_origin"],
                           prob["dsm_gsd"])
    # validity flags: exact, except for pixels whose map position is within fp noise of the heightfield border
    assert (got[:, 3] == want[:, 3]).mean() >= 0.999 and set(np.unique(got[:, 3])) <= {0.0, 1.0}
    same = got[:, 3] == want[:, 3]
    assert np.abs(got[same, :2] - want[same, :2]).max() <= 6.2e-5
    # D^r: the bilinear sample is evaluated at double-precision map coordinates on both sides
    assert np.abs(got[same, 2] - want[same, 2]).max() <= 1e-4
    # the crop corners land on the footprint corners
    assert np.abs(got[:4, :2] - c_np[:, :2]).max() <= 1e-3
    assert (got[:, 3] == 1).mean() > 0.5
    # the anchors are what pilot_refine_inputs.points_dev takes: refine against them, GPU vs oracle on the same anchors
    u, v, _ = wl.project(prob["gt_pose"].reshape(3, 4), K, got[:, :3].astype(np.float64))
    q = dict(prob)
    q["points"] = [got] * 3
    q["ref_feat"] = [prob["ref_feat"][l][:1].repeat(got.shape[0], 0) for l in range(3)]
    q["params"] = dict(prob["params"], min_valid=8)
    gpu = binding.refine(q)
    orc = po.run(po.Bound(q), n_threads=8)
    eH, eg, ec = parity.system_errors(gpu, orc, 0)
    assert max(eH.max(), eg.max(), ec.max()) <= 5e-3
    # anchors of weight 0 contribute nothing: dropping them leaves the system unchanged
    keep = got[:, 3] == 1
    q2 = dict(q)
    q2["points"] = [got[keep]] * 3
    q2["ref_feat"] = [r[keep] for r in q["ref_feat"]]
    g2 = binding.refine(q2)
    assert np.allclose(g2["iter_hessian"][0], gpu["iter_hessian"][0], rtol=1e-4, atol=1e-3 * np.abs(gpu["iter_hessian"][0]).max())


def test_lift_with_degenerate_footprint_gives_weight_zero():
    import torch
    from paper_2606_31098_b200 import binding
    prob, K, W, H = scene()
    corners = dev(np.full((4, 4), np.nan))
    pts = binding.lift_anchors(corners, 64, 64, dev(np.zeros((5, 2))), dev(prob["dsm"]), prob["dsm_origin"], prob["dsm_gsd"])
    torch.cuda.synchronize()
    assert np.all(pts.cpu().numpy() == 0)
    corners = dev(np.zeros((4, 4)))                               # all four corners coincide: singular system
    pts = binding.lift_anchors(corners, 64, 64, dev(np.ones((5, 2))), dev(prob["dsm"]), prob["dsm_origin"], prob["dsm_gsd"])
    torch.cuda.synchronize()
    assert np.all(pts.cpu().numpy()[:, 3] == 0)

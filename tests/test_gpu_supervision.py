"""pilot_refine_reprojection_loss (supp Eq.7-8) through the C-ABI against oracle/pilot_supervision.py."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _scene(seed, n_points, n_poses):
    from tests.small_problems import look_down_pose
    rng = np.random.default_rng(seed)
    pts = np.column_stack([rng.uniform(-120, 120, n_points), rng.uniform(-120, 120, n_points), rng.uniform(0, 30, n_points),
                           np.ones(n_points)]).astype(np.float32)
    T = np.asarray(look_down_pose(np.array([0.0, -110.0, 140.0]), 50.0), np.float64).reshape(3, 4)
    poses = []
    for k in range(n_poses):
        w = rng.uniform(-0.15, 0.15, 3) * (k > 0)
        th = np.linalg.norm(w)
        Kx = np.array([[0, -w[2], w[1]], [w[2], 0, -w[0]], [-w[1], w[0], 0]])
        E = np.eye(3) + (np.sin(th) / th * Kx + (1 - np.cos(th)) / th ** 2 * Kx @ Kx if th > 0 else 0)
        Tk = np.hstack([T[:, :3] @ E, (T[:, 3] + rng.uniform(-12, 12, 3) * (k > 0))[:, None]])
        poses.append(Tk.reshape(-1))
    return pts, T.reshape(-1).astype(np.float32), np.asarray(poses, np.float32)


@pytest.mark.parametrize("alpha", [2.0, 1.0, 0.0, -2.0, -np.inf, 0.5])
@pytest.mark.parametrize("n_points", [1, 255, 4099])
def test_reprojection_loss_matches_oracle(alpha, n_points):
    import torch
    from oracle import pilot_supervision as ps
    from paper_2606_31098_b200 import binding
    pts, Ts, poses = _scene(11 + n_points, n_points, 37)
    K = (420.0, 415.0, 319.5, 239.5)
    L, n = binding.reprojection_loss(torch.from_numpy(poses).cuda(), Ts, torch.from_numpy(pts).cuda(), K, 640, 480, 0.1, alpha, 2.5)
    Lo, no = ps.reprojection_loss(poses, Ts, pts, K, 640, 480, 0.1, alpha, 2.5)
    assert np.array_equal(n.cpu().numpy(), no)                       # the visible set is decided in double on both sides
    assert np.allclose(L.cpu().numpy(), Lo, rtol=2e-6, atol=1e-12)   # double arithmetic, one rounding to fp32 at the end
    assert L[0].item() == 0.0 and (n_points < 200 or no[0] > 0)      # pose 0 is the ground truth


def test_reprojection_loss_edge_cases_and_errors():
    import ctypes as C
    import torch
    from paper_2606_31098_b200 import binding
    pts, Ts, poses = _scene(5, 300, 4)
    K = (420.0, 415.0, 319.5, 239.5)
    dp, dpts = torch.from_numpy(poses).cuda(), torch.from_numpy(pts).cuda()
    L, n = binding.reprojection_loss(dp, Ts, dpts[:0].contiguous(), K, 640, 480, 0.1, 1.0, 1.0)      # no points
    assert torch.all(L == 0) and torch.all(n == 0)
    behind = dpts.clone(); behind[:, 2] = 500.0                                                     # above the camera
    L, n = binding.reprojection_loss(dp, Ts, behind, K, 640, 480, 0.1, 1.0, 1.0)
    assert torch.all(L == 0) and torch.all(n == 0)
    L, n = binding.reprojection_loss(dp[:0].contiguous(), Ts, dpts, K, 640, 480, 0.1, 1.0, 1.0)      # no poses
    assert L.numel() == 0
    a, b = binding.reprojection_loss(dp, Ts, dpts, K, 640, 480, 0.1, -2.0, 3.0), binding.reprojection_loss(dp, Ts, dpts, K, 640, 480, 0.1, -2.0, 3.0)
    assert torch.equal(a[0], b[0])                                                                  # deterministic
    for bad in (dict(alpha=float("nan")), dict(alpha=float("inf")), dict(scale=0.0), dict(width=0)):
        kw = dict(alpha=1.0, scale=1.0, width=640); kw.update(bad)
        with pytest.raises(RuntimeError):
            binding.reprojection_loss(dp, Ts, dpts, K, kw["width"], 480, 0.1, kw["alpha"], kw["scale"])


def test_supervision_of_an_unrolled_refinement_decreases():
    """The use the paper makes of it: the loss after the unrolled LM steps of a refinement that converges goes down
    (config 0: 2 deg / 2 m perturbation, 0 ... 5 steps)."""
    import torch
    from oracle import pilot_supervision as ps
    from paper_2606_31098_b200 import binding
    from paper_2606_31098_b200 import workloads as wl
    prob = wl.config0()
    steps = []
    for k in range(0, 6):
        out = binding.refine(prob, dict(prob["params"], iters=[k]))
        steps.append(np.asarray(out["poses"], np.float32).reshape(-1, 12)[0])
    poses = np.asarray(steps, np.float32)
    pts = np.ascontiguousarray(prob["points"][0], np.float32)
    K = prob["intrinsics"][0]
    Ts = np.asarray(prob["gt_pose"], np.float32)
    L, n = binding.reprojection_loss(torch.from_numpy(poses).cuda(), Ts, torch.from_numpy(pts).cuda(), K, 64, 48, 0.1, 1.0, 1.0)
    Lo, no = ps.reprojection_loss(poses, Ts, pts, K, 64, 48, 0.1, 1.0, 1.0)
    assert np.array_equal(n.cpu().numpy(), no) and np.allclose(L.cpu().numpy(), Lo, rtol=2e-6, atol=1e-12)
    assert no[0] > 100 and Lo[0] > 0.1 and Lo[-1] < 0.05 * Lo[0]


def test_backward_pieces_match_the_oracle():
    """Pose gradient of the reprojection loss and the adjoint of LM steps taken from a real run's records (config 0),
    against oracle/pilot_supervision.py (itself pinned by central differences): double arithmetic on both sides, one
    rounding to fp32 on the GPU's outputs."""
    import torch
    from oracle import pilot_oracle as po
    from oracle import pilot_supervision as ps
    from paper_2606_31098_b200 import binding, workloads as wl
    prob = wl.config0()
    orc = po.run(po.Bound(prob, dict(iters=[6])))
    poses = np.concatenate([prob["init_poses"][:1], orc["iter_poses"][1:, 0].astype(np.float32), orc["poses"][:1]])
    pts = prob["points"][0]
    K, W, H = prob["intrinsics"][0], prob["width"][0], prob["height"][0]
    d = torch.device("cuda")
    for alpha, c in [(1.0, 2.0), (2.0, 1.0), (0.0, 3.0), (-2.0, 1.5), (-np.inf, 4.0)]:
        L, nv, G = binding.reprojection_loss_grad(torch.from_numpy(poses).to(d), prob["gt_pose"], torch.from_numpy(pts).to(d), K, W, H,
                                                  0.1, alpha, c)
        Lo, no, Go = ps.reprojection_loss_grad(poses, np.asarray(prob["gt_pose"], np.float32), pts, K, W, H, 0.1, alpha, c)
        assert np.array_equal(nv.cpu().numpy(), no) and no.min() > 50
        assert np.allclose(L.cpu().numpy(), Lo, rtol=2e-6, atol=1e-12)
        assert np.allclose(G.cpu().numpy(), Go, rtol=2e-6, atol=2e-6 * np.abs(Go).max())
    # the recorded systems of the run, the gradient of L at the pose each step produced
    Hs, gs, lam = orc["iter_hessian"][:, 0], orc["iter_gradient"][:, 0], orc["iter_lambda"][:, 0]
    nxt = np.concatenate([orc["iter_poses"][1:, 0], orc["poses64"][:1]]).astype(np.float32)
    q = ps.reprojection_loss_grad(nxt, np.asarray(prob["gt_pose"], np.float32), pts, K, W, H, 0.1, 1.0, 2.0)[2].astype(np.float32)
    for damp in ("identity", "diag"):
        o = binding.lm_step_adjoint(torch.from_numpy(Hs).to(d), torch.from_numpy(gs).to(d), torch.from_numpy(lam).to(d),
                                    torch.from_numpy(q).to(d), damp)
        o = {k: v.cpu().numpy() for k, v in o.items()}
        assert np.all(o["status"] == 0)
        for m in range(Hs.shape[0]):
            dxi, GH, Gg, qp = ps.lm_step_adjoint(Hs[m].astype(np.float64), gs[m].astype(np.float64), float(lam[m]), damp == "diag",
                                                 q[m].astype(np.float64))
            assert np.allclose(o["dxi"][m], dxi, rtol=1e-5, atol=1e-6 * np.abs(dxi).max())
            assert np.allclose(o["grad_gradient"][m], Gg, rtol=1e-5, atol=1e-6 * np.abs(Gg).max())
            assert np.allclose(o["grad_hessian"][m].reshape(6, 6), GH, rtol=1e-5, atol=1e-6 * np.abs(GH).max())
            assert np.allclose(o["q_prev"][m], qp, rtol=1e-5, atol=1e-6 * np.abs(qp).max())
    # a system that is not positive definite is flagged, not an error return
    bad = binding.lm_step_adjoint(torch.from_numpy(-Hs[:1]).to(d), torch.from_numpy(gs[:1]).to(d), torch.zeros(1, device=d),
                                  torch.from_numpy(q[:1]).to(d))
    assert int(bad["status"].cpu().numpy()[0]) == 4

"""Pins of oracle/pilot_hypotheses.py against what the paper and the mathematics fix (CPU only)."""
import itertools
import os

import numpy as np
from scipy.linalg import expm
from scipy.spatial.transform import Rotation

from oracle import pilot_hypotheses as ph
from oracle import pilot_oracle as po
from tests.small_problems import tiny

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_counts.txt")
PAPER_YAWS = [-9, -7, -5, -3, -1, 1, 3, 5, 7, 9]          # supp Eq.(4)


def golden_counts():
    out = {}
    for line in open(GOLDEN):
        if line.strip() and not line.startswith("#"):
            v, name = line.split()[:2]
            out[name] = int(v)
    return out


def skew(w):
    return np.array([[0, -w[2], w[1]], [w[2], 0, -w[0]], [-w[1], w[0], 0.0]])


def test_grid_has_the_papers_1210_entries():
    g = ph.grid_offsets(10.0, 2.0, PAPER_YAWS, [0, 0, 1.0])
    assert g.shape == (golden_counts()["initial_hypotheses"], 6) == (1210, 6)
    # 11 x 11 translations, step 2 m, range +-10 m; no z offset; 10 yaw values, none of them zero
    assert sorted(set(g[:, 3])) == sorted(set(g[:, 4])) == [-10, -8, -6, -4, -2, 0, 2, 4, 6, 8, 10]
    assert np.all(g[:, 5] == 0) and np.all(g[:, :2] == 0)
    assert np.allclose(sorted(set(np.rad2deg(g[:, 2]).round(6))), PAPER_YAWS)
    assert len({tuple(r) for r in g.round(9)}) == 1210                            # a Cartesian product: all distinct
    # ordering: x slowest, then y, yaw fastest
    assert np.allclose(g[0], [0, 0, np.deg2rad(-9), -10, -10, 0])
    assert np.allclose(g[9], [0, 0, np.deg2rad(9), -10, -10, 0])
    assert np.allclose(g[10], [0, 0, np.deg2rad(-9), -10, -8, 0])
    assert np.allclose(g[110], [0, 0, np.deg2rad(-9), -8, -10, 0])
    assert np.allclose(g[-1], [0, 0, np.deg2rad(9), 10, 10, 0])


def test_seed_rotation_is_the_matrix_exponential():
    rng = np.random.default_rng(1)
    T = np.concatenate([Rotation.random(random_state=2).as_matrix(), rng.normal(size=(3, 1)) * 50], 1)
    off = rng.normal(size=(7, 6)) * [0.2, 0.2, 0.2, 5, 5, 5]
    off[0] = 0
    cam = ph.seed_hypotheses(T.reshape(-1), off, ph.SEED_CAMERA).reshape(-1, 3, 4)
    wor = ph.seed_hypotheses(T.reshape(-1), off, ph.SEED_WORLD).reshape(-1, 3, 4)
    assert np.array_equal(cam[0], T) and np.array_equal(wor[0], T)                # zero offset = the prior itself
    for m in range(7):
        E = expm(skew(off[m, :3]))                                                # textbook routine
        assert np.allclose(cam[m][:, :3], T[:, :3] @ E, atol=1e-13)
        assert np.allclose(wor[m][:, :3], E @ T[:, :3], atol=1e-13)
        assert np.allclose(cam[m][:, 3], T[:, 3] + off[m, 3:]) and np.allclose(wor[m][:, 3], T[:, 3] + off[m, 3:])
        assert np.allclose(cam[m][:, :3].T @ cam[m][:, :3], np.eye(3), atol=1e-13)


def test_camera_frame_offsets_follow_the_workload_convention():
    """workloads.perturbed_poses: R_wc_m = R_wc_gt Rot(d), C_m = C_gt + t — the SEED_CAMERA composition."""
    from paper_2606_31098_b200 import workloads as wl
    T = wl.pitched_pose([3.0, -40.0, 120.0], 50.0, 20.0)
    rng = np.random.Generator(np.random.PCG64(5))
    poses = wl.perturbed_poses(rng, T, 6, 5.0, 10.0, first_is_gt=True)
    rng = np.random.Generator(np.random.PCG64(5))                                 # replay the generator's draws
    off = np.zeros((6, 6))
    for m in range(6):
        off[m, :3] = np.deg2rad(rng.uniform(-5.0, 5.0, 3))
        off[m, 3:] = rng.uniform(-10.0, 10.0, 3)
    off[0] = 0
    mine = ph.seed_hypotheses(T.reshape(-1), off, ph.SEED_CAMERA)
    assert np.allclose(mine, poses, atol=1e-5)


def test_world_yaw_leaves_the_gravity_residual_unchanged():
    """yaw is not constrained by gravity. A SEED_WORLD offset about the vertical changes R_cw but not
    R_cw gamma^W, so Eq.(3)'s residual (computed by the refinement oracle) is identical for every yaw hypothesis."""
    prob = tiny(seed=3)
    b = po.Bound(prob, dict(w_gravity=1.0))
    up = -np.asarray(prob["gravity_world"], np.float64)
    g = ph.grid_offsets(4.0, 2.0, PAPER_YAWS, up)
    poses = ph.seed_hypotheses(prob["gt_pose"], g, ph.SEED_WORLD).reshape(-1, 3, 4)
    r0, _ = po.gravity(b, po.pose_to_RC(prob["gt_pose"])[0])
    headings = set()
    for T in poses:
        r, _ = po.gravity(b, po.pose_to_RC(T)[0])
        assert np.allclose(r, r0, atol=1e-13)
        headings.add(round(float(np.arctan2(T[0, 2], T[1, 2])), 9))
    assert len(headings) == len(PAPER_YAWS)                                       # but the heading does change
    # a camera-frame offset about the camera z axis does change it (the tilt moves): the two frames differ
    cam = ph.seed_hypotheses(prob["gt_pose"], [[0, 0, 0.1, 0, 0, 0]], ph.SEED_CAMERA).reshape(3, 4)
    r, _ = po.gravity(b, po.pose_to_RC(cam)[0])
    assert np.abs(r - r0).max() > 1e-3


def test_select_best_rules():
    assert ph.select_best([3.0, 1.0, 2.0]) == 1
    assert ph.select_best([3.0, 1.0, 1.0, 0.5, 0.5]) == 3                         # ties -> lowest index
    assert ph.select_best([np.nan, np.inf, 7.0, np.nan]) == 2                     # NaN = +inf
    assert ph.select_best([np.inf, np.inf]) == 0
    assert ph.select_best([np.nan, np.nan]) == 0


def test_topk_against_brute_force():
    rng = np.random.default_rng(9)
    for n, k in [(1, 1), (5, 3), (7, 7), (9, 4)]:
        c = rng.integers(0, 4, n).astype(np.float64)                              # many ties
        if n > 4:
            c[1] = np.nan; c[3] = np.inf
        got = ph.prune_topk(c, k)
        key = [(np.inf if np.isnan(v) else v, i) for i, v in enumerate(c)]
        # brute force: the unique k-subset + order whose (cost, index) sequence is lexicographically smallest
        best = min(itertools.permutations(range(n), k), key=lambda p: [key[i] for i in p])
        assert list(got) == list(best)
    c = rng.normal(size=1210)
    t = ph.prune_topk(c, golden_counts()["retained_hypotheses"])
    assert len(t) == 128 and len(set(t)) == 128
    assert np.array_equal(c[t], np.sort(c)[:128])                                 # library routine
    assert ph.select_best(c) == t[0]

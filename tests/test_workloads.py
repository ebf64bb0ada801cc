"""Host-side checks of the seeded workload generators (no GPU, no method arithmetic)."""
import os

import numpy as np

from paper_2606_31098_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_counts.txt")


def golden():
    out = {}
    for line in open(GOLDEN):
        if line.strip() and not line.startswith("#"):
            v, name = line.split()[:2]
            out[name] = int(v)
    return out


def test_paper_counts_arithmetic():
    g = golden()
    assert g["initial_hypotheses"] == 11 * 11 * 10
    per_frame = g["geo_anchors"] * (g["initial_hypotheses"] * g["iters_coarse"] +
                                    g["retained_hypotheses"] * (g["iters_medium"] + g["iters_fine"]))
    assert per_frame == g["point_hyp_iters_per_frame"]
    p = wl.paper_frame()
    assert p["units"] == per_frame and p["keep"] == g["retained_hypotheses"]
    assert p["channels"] == [g["descriptor_channels"]] * 3 and p["points"][0].shape[0] == g["geo_anchors"]
    assert p["params"]["iters"] == [g["iters_coarse"], g["iters_medium"], g["iters_fine"]]
    assert len(wl.PAPER_YAWS) == 10 and 0.0 not in wl.PAPER_YAWS
    assert g["unrolled_training_steps"] == g["iters_coarse"] + g["iters_medium"] + g["iters_fine"]   # PAPER.md:440 and :205 agree


def test_paper_frame_is_normalised_and_weighted():
    p = wl.paper_frame()
    for l in range(3):
        q = wl.decode(p["query_feat"][l], p["dtype"]).astype(np.float64)
        assert np.abs(np.linalg.norm(q, axis=-1) - 1).max() < 1e-2                   # bf16 rounding of a unit vector
        c = p["query_conf"][l]
        assert c.shape == (p["height"][l], p["width"][l]) and 0 < c.min() and c.max() < 1
    assert 0.5 <= p["points"][0][:, 3].min() and p["points"][0][:, 3].max() <= 1.0
    # the prior differs from the ground truth by a yaw about the vertical and a horizontal shift only
    Tg, Tp = p["gt_pose"].reshape(3, 4), p["prior_pose"].reshape(3, 4).astype(np.float64)
    assert abs(Tp[2, 3] - Tg[2, 3]) < 1e-4 and np.allclose(Tp[:2, 3] - Tg[:2, 3], [3.1, -4.3], atol=1e-4)
    D = Tp[:, :3] @ Tg[:, :3].T
    assert np.allclose(D[2], [0, 0, 1], atol=1e-6) and np.isclose(np.rad2deg(np.arctan2(D[1, 0], D[0, 0])), 2.2, atol=1e-3)


def test_configs_have_baseline_shapes():
    p = wl.config0()
    assert (p["width"], p["height"], p["channels"], p["dtype"]) == ([64], [48], [16], "f32")
    assert p["points"][0].shape == (256, 4) and p["init_poses"].shape == (1, 12) and p["units"] == 1280
    p = wl.config1()
    assert p["width"] == [120, 240, 480] and p["height"] == [68, 135, 270] and p["channels"] == [32] * 3
    assert p["init_poses"].shape == (64, 12) and p["units"] == 3 * 64 * 4096 * 10 and p["dsm"].shape == (512, 512)
    assert np.array_equal(p["init_poses"][0], p["gt_pose"].astype(np.float32))       # hypothesis 0 = GT
    q = wl.config1()
    assert all(np.array_equal(a, b) for a, b in zip(p["query_feat"], q["query_feat"]))   # seeded: reproducible


def test_config3_sequence_frames():
    seq = wl.Config3Sequence(n_frames=300)
    assert seq.dsm.shape == (2048, 2048) and seq.offsets.shape == (128, 6) and np.all(seq.offsets[0] == 0)
    assert np.abs(np.rad2deg(seq.offsets[:, :3])).max() <= 5 and np.abs(seq.offsets[:, 3:]).max() <= 10
    assert seq.units_per_frame == 15728640
    # trajectory: 0.5 m per frame (15 m/s at 30 fps), 150 m above the mean terrain, pitch within 30-60 deg
    C = np.stack([seq.gt_pose(i)[:, 3] for i in range(300)])
    assert np.allclose(np.linalg.norm(np.diff(C, axis=0), axis=1), 0.5, atol=1e-3)
    assert np.allclose(C[:, 2], seq.z_mean + 150.0)
    pitch = np.array([np.rad2deg(np.arcsin(-seq.gt_pose(i)[2, 2])) for i in range(300)])
    assert 29.9 <= pitch.min() and pitch.max() <= 60.1
    f = seq.frame(7)
    assert f["width"] == [120, 240, 480] and f["dtype"] == "bf16" and f["points"][0].shape == (4096, 4)
    assert "init_poses" not in f and f["units"] == seq.units_per_frame
    g = seq.frame(7)
    assert np.array_equal(f["query_feat"][2], g["query_feat"][2]) and f["range_meas"] == g["range_meas"]
    assert not np.array_equal(f["query_feat"][2], seq.frame(8)["query_feat"][2])      # new field per frame
    # a usable share of the anchors projects into the image at the ground-truth pose
    u, v, Z = wl.project(seq.gt_pose(7), seq.K, f["points"][0][:, :3].astype(np.float64))
    assert ((u >= 0) & (u < 479) & (v >= 0) & (v < 269) & (Z > 0)).mean() > 0.3
    fr = list(seq.frames(indices=[7, 8], workers=2))
    assert np.array_equal(fr[0]["query_feat"][1], f["query_feat"][1]) and fr[1]["frame"] == 8

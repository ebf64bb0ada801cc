"""Config 3 (BASELINE.json configs[3]): the 300-frame streaming sequence through pilot_refine_sequence_*.
Parity is frame-local: frames 0-4 are chained on the oracle side too (its own seeds, its own
arg-min); afterwards every 50th frame the oracle is fed the GPU's seed poses of that frame and both refine them."""
import numpy as np
import pytest

from tests import parity

pytestmark = pytest.mark.gpu

TOL = 5e-3   # bf16 features: 5e-3 rad / 5e-3 m (north_star)


def make_sequence(seq, n_frames):
    from paper_2606_31098_b200 import binding
    L = seq.LEVELS
    return binding.Sequence(3, [l[0] for l in L], [l[1] for l in L], [l[2] for l in L], "bf16", seq.H, seq.N,
                            sum(seq.iters), seq.offsets, seq.dsm, seq.origin, seq.gsd, seq.gravity_world, n_frames)


def oracle_frame(frame, seeds):
    from oracle import pilot_oracle as po
    from paper_2606_31098_b200 import workloads as wl
    return po.run(po.Bound(wl.with_poses(frame, seeds)), n_threads=16)


def test_config3_streaming_sequence():
    import torch
    from oracle import pilot_hypotheses as ph
    from paper_2606_31098_b200 import workloads as wl
    n_frames = 300
    seq = wl.Config3Sequence(n_frames=n_frames)
    S = make_sequence(seq, n_frames)
    S.set_prior(seq.gt_pose(0).reshape(-1))
    checked = [0, 1, 2, 3, 4] + list(range(50, n_frames, 50)) + [n_frames - 1]
    kept, gpu_sets = {}, {}
    gen = seq.frames()
    nxt = next(gen)
    S.upload(nxt)
    for i in range(n_frames):
        cur = nxt
        if i + 1 < n_frames:
            nxt = next(gen)
            S.upload(nxt)                      # frame i+1 copies while frame i refines
        S.step(seq.params)
        assert S.last_launches == 1 + 3 + 3            # AUTO: one cluster-resident launch per level at this size
        if i in checked:
            kept[i] = cur
            gpu_sets[i] = S.last_frame()       # synchronises: test only
    rows = S.results()
    torch.cuda.synchronize()
    S.close()

    # ---- frames 0-4: the oracle runs its own chain from the same prior
    prior = seq.gt_pose(0).reshape(-1).astype(np.float32).astype(np.float64)
    for i in range(5):
        seeds = ph.seed_hypotheses(prior, seq.offsets, ph.SEED_CAMERA)
        orc = oracle_frame(kept[i], seeds)
        b = ph.select_best(orc["cost64"])
        gb = int(rows[i, 13])
        # most hypotheses reach the same optimum, so WHICH of them has the lowest cost is decided by rounding:
        # compare what is unique (the selected pose and objective) and check that the GPU's choice is valid
        assert parity.rot_angle(rows[i, :12], orc["poses64"][b])[0] <= TOL
        assert parity.trans_dist(rows[i, :12], orc["poses64"][b])[0] <= TOL
        assert abs(rows[i, 12] - orc["cost64"][b]) <= 5e-3 * orc["cost64"][b]
        assert abs(orc["cost64"][gb] - orc["cost64"][b]) <= 5e-3 * orc["cost64"][b]
        assert abs(int(rows[i, 14]) - orc["n_valid"][gb]) <= 2
        assert rows[i, 12] == gpu_sets[i][2].min() and gpu_sets[i][2][gb] == rows[i, 12]
        assert gb == int(np.argmin(gpu_sets[i][2]))
        # frame 0: the same prior on both sides, so the GPU seeds are the oracle's to fp32 rounding; later frames are
        # seeded from each side's own previous estimate, which agree to the pose tolerance
        assert np.abs(gpu_sets[i][0] - seeds).max() <= (4e-5 if i == 0 else 2 * TOL)
        prior = orc["poses64"][b].astype(np.float32).astype(np.float64)     # the estimate crosses the API as fp32

    # ---- every 50th frame: the oracle refines the GPU's own seeds of that frame
    for i in checked[5:]:
        seeds, poses, cost = gpu_sets[i]
        orc = oracle_frame(kept[i], seeds)
        g = dict(poses=poses, cost=cost)
        conv = parity.converged(orc, step_tol=5e-4)       # 200-400 m ranges: last accepted steps are ~1e-5..1e-4 m
        er, et = parity.pose_errors(g, orc)
        # Whether the ORACLE ends a frame on a tiny accepted step depends on the seeds to the last bit (on some frames an
        # anchor at the border of the map makes it reject every step after one of ~1e-3 m, for most hypotheses at once),
        # and the seeds are the GPU's own estimate of the previous frame: the size of the flagged set is a property of
        # the frame, not of the path under test. What is asserted: every flagged hypothesis agrees, the set is not empty,
        # and at least half of ALL hypotheses agree with the oracle whatever it flagged ("report the
        # matching fraction of the rest").
        assert conv.any(), i
        assert er[conv].max() <= TOL and et[conv].max() <= TOL, (i, er[conv].max(), et[conv].max())
        assert ((er <= TOL) & (et <= TOL)).sum() >= seq.H // 2, (i, ((er <= TOL) & (et <= TOL)).sum())
        b = ph.select_best(orc["cost64"])
        assert er[b] <= TOL and et[b] <= TOL
        gb = int(rows[i, 13])
        assert abs(cost[gb] - orc["cost64"][b]) <= 5e-3 * orc["cost64"][b]
        assert np.array_equal(rows[i, :12], poses[gb]) and rows[i, 12] == cost[gb]

    # ---- properties over the whole sequence: the track follows the ground truth (noise-limited)
    gt = np.stack([seq.gt_pose(i).reshape(-1) for i in range(n_frames)])
    er, et = parity.rot_angle(rows[:, :12], gt), parity.trans_dist(rows[:, :12], gt)
    assert np.isfinite(rows[:, 12]).all()
    assert np.rad2deg(er).max() < 0.5 and et.max() < 1.5, (np.rad2deg(er).max(), et.max())
    assert np.all(rows[:, 15] == 0)            # status of every selected hypothesis is clean


def test_sequence_argument_errors():
    from paper_2606_31098_b200 import binding, workloads as wl
    seq = wl.Config3Sequence(n_frames=3, H=8, N=512, iters=(1, 1, 1))
    S = make_sequence(seq, 2)
    with pytest.raises(RuntimeError, match="-1"):
        S.step(seq.params)                      # nothing uploaded
    f = seq.frame(0)
    S.upload(f); S.upload(f)
    with pytest.raises(RuntimeError, match="-3"):
        S.upload(f)                             # both halves pending
    S.set_prior(seq.gt_pose(0).reshape(-1))
    S.step(seq.params); S.step(seq.params)
    S.upload(f)
    with pytest.raises(RuntimeError, match="-1"):
        S.step(seq.params)                      # log full
    r = S.results()
    assert r.shape == (2, 16) and np.isfinite(r).all()
    # same frame, second step seeded from the first estimate: still at the same optimum
    assert parity.trans_dist(r[0, :12], r[1, :12])[0] < 0.05
    S.close()


def test_pinned_frames_are_copied_directly_and_give_the_same_track():
    from paper_2606_31098_b200 import binding, workloads as wl
    seq = wl.Config3Sequence(n_frames=6, H=16, N=1024, iters=(2, 2, 2))
    tracks = []
    for pin in (False, True):
        S = make_sequence(seq, 6)
        S.set_prior(seq.gt_pose(0).reshape(-1))
        frames = [binding.make_frame(seq.frame(i), pin=pin) for i in range(6)]
        S.upload(frames[0])
        for i in range(6):
            if i + 1 < 6:
                S.upload(frames[i + 1])
            S.step(seq.params)
        tracks.append(S.results())
        S.close()
    assert np.array_equal(tracks[0], tracks[1])

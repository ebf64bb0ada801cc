"""pilot_refine_sort_anchors against its oracle (bit-exact permutation: index work), and a refinement on shuffled anchors:
the sums do not depend on the order (Eq.2, Eq.8 are sums over j), so GPU-on-sorted == oracle-on-shuffled within tolerance."""
import numpy as np
import pytest

from oracle import pilot_anchor_order as ao
from paper_2606_31098_b200 import workloads as wl
from tests import parity

pytestmark = pytest.mark.gpu


def _sort(points, ref, channels, dtype):
    import torch
    from paper_2606_31098_b200 import binding
    prob = dict(n_levels=1, dtype=dtype, width=[8], height=[8], channels=[channels], query_feat=[np.zeros((8, 8, channels), np.float32 if dtype == "f32" else np.uint16)],
                intrinsics=[(1, 1, 0, 0)], points=[points], ref_feat=[ref], init_poses=None, gravity_world=np.zeros(3),
                gravity_imu=np.zeros(3), range_ray_cam=np.zeros(3), range_meas=0.0, dsm=None, dsm_origin=(0, 0), dsm_gsd=1.0)
    di = binding.DeviceInputs(prob, 0)
    perm = di.sort_anchors()[0]
    torch.cuda.synchronize()
    n = points.shape[0]
    row = channels * (4 if dtype == "f32" else 2)
    pts = np.frombuffer(bytes(di.keep[-2].cpu().numpy()), np.float32).reshape(n, 4)
    rf = np.frombuffer(bytes(di.keep[-1].cpu().numpy()), np.uint8).reshape(n, row)
    return perm.cpu().numpy(), pts, rf


@pytest.mark.parametrize("n", [1, 31, 1000, 65536, 100003])
def test_permutation_is_bit_identical_with_the_oracle(n):
    rng = np.random.default_rng(n)
    P = np.zeros((n, 4), np.float32)
    P[:, :2] = rng.uniform(-511.7, 733.1, (n, 2))
    P[:, 2], P[:, 3] = rng.uniform(0, 40, n), rng.uniform(0.5, 1, n)
    if n >= 1000:
        P[5:25, :2] = P[5, :2]                       # ties keep their input order
        P[77, 0] = np.nan                            # a non-finite anchor gets key component 0 and does not move the box
    ref = rng.integers(0, 65535, (n, 32), dtype=np.uint16)
    perm, pts, rf = _sort(P, ref, 32, "bf16")
    want = ao.morton_order(P)
    assert np.array_equal(perm, want)
    assert np.array_equal(pts.view(np.uint32), P[want].view(np.uint32))
    assert np.array_equal(rf, ref[want].view(np.uint8).reshape(n, -1))


def test_degenerate_boxes_and_arguments():
    from paper_2606_31098_b200 import binding
    P = np.zeros((100, 4), np.float32); P[:, 0] = 3.0; P[:, 1] = np.arange(100) % 7       # x extent 0
    perm, _, _ = _sort(P, np.zeros((100, 8), np.float32), 8, "f32")
    assert np.array_equal(perm, ao.morton_order(P))
    L = binding.lib()
    assert L.pilot_refine_sort_anchors_temp_bytes(0) == 0 and L.pilot_refine_sort_anchors_temp_bytes(4096) >= 5 * 4096
    assert L.pilot_refine_sort_anchors(None, None, 5, 8, 0, None, None, None, None, 0, None) == -1


def test_refinement_on_device_sorted_anchors_matches_oracle_on_shuffled_input():
    import torch
    from oracle import pilot_oracle as po
    from paper_2606_31098_b200 import binding
    prob = wl.config1(H=12, N=3000, iters=(3, 3, 3))
    rng = np.random.default_rng(5)
    for l in range(prob["n_levels"]):
        perm = rng.permutation(prob["points"][l].shape[0])
        prob["points"][l] = np.ascontiguousarray(prob["points"][l][perm])
        prob["ref_feat"][l] = np.ascontiguousarray(prob["ref_feat"][l][perm])
    orc = po.run(po.Bound(prob), n_threads=8)
    di = binding.DeviceInputs(prob, 0)
    di.sort_anchors()
    r = binding.Refiner.for_inputs(di, prob["params"], 0)
    out = r.run(di, prob["params"])
    torch.cuda.synchronize()
    gpu = {k: v.cpu().numpy() for k, v in out.items()}
    r.close()
    eH, eg, ec = parity.system_errors(gpu, orc, 0)
    assert eH.max() < 5e-3 and eg.max() < 5e-3 and ec.max() < 5e-3
    conv = parity.converged(orc)
    er, et = parity.pose_errors(gpu, orc)
    assert conv.sum() >= 6 and er[conv].max() < 5e-3 and et[conv].max() < 5e-3

"""Tiny random problems for the oracle pins (test-side only; no method arithmetic beyond scene placement)."""
import numpy as np
from scipy.spatial.transform import Rotation


def look_down_pose(C, pitch_deg=60.0):
    p = np.deg2rad(pitch_deg)
    f = np.array([0.0, np.cos(p), -np.sin(p)])
    right = np.cross(f, [0, 0, 1.0]); right /= np.linalg.norm(right)
    down = np.cross(f, right)
    T = np.zeros((3, 4))
    T[:, 0], T[:, 1], T[:, 2], T[:, 3] = right, down, f, C
    return T


def tiny(seed=0, N=12, C=3, W=40, H=30, n_hyp=1, dtype="f32", conf=False, affine=False, dsm_plane=None,
         smooth=True, origin_shift=(0.0, 0.0, 0.0)):
    """One-level problem: random (or affine) feature map, points on a gentle heightfield under the camera."""
    rng = np.random.default_rng(seed)
    sh = np.asarray(origin_shift, np.float64)
    ys, xs = np.mgrid[0:H, 0:W].astype(np.float64)
    if affine:
        a, b, d = rng.normal(size=C), rng.normal(size=C) * 0.1, rng.normal(size=C) * 0.1
        F = a + b * xs[..., None] + d * ys[..., None]
        aff = (a, b, d)
    else:
        F = rng.normal(size=(H, W, C))
        if smooth:  # low-pass so finite differences stay in one bilinear cell comfortably
            for _ in range(2):
                F = 0.25 * (F + np.roll(F, 1, 0) + np.roll(F, 1, 1) + np.roll(np.roll(F, 1, 0), 1, 1))
        aff = None
    Wd = Hd = 33
    gsd = 2.0
    origin = np.array([-32.0, -32.0])
    gy, gx = np.mgrid[0:Hd, 0:Wd].astype(np.float64)
    if dsm_plane is not None:
        h0, pa, pb = dsm_plane   # z = h0 + pa*x + pb*y in world metres (before the origin shift)
        dsm = h0 + pa * (origin[0] + gx * gsd) + pb * (origin[1] + gy * gsd)
    else:
        dsm = 3.0 * np.sin(gx / 5.0) * np.cos(gy / 7.0) + 5.0
    T = look_down_pose(np.array([0.0, -40.0, 75.0]))
    K = (30.0, 32.0, W / 2.0 - 0.3, H / 2.0 + 0.2)
    px = rng.uniform(-18, 18, N); py = rng.uniform(-14, 14, N)
    pz = 5.0 + rng.uniform(-2, 2, N)
    P = np.stack([px, py, pz, rng.uniform(0.5, 1.5, N) if conf else np.ones(N)], 1)
    P[:, :3] += sh
    T[:, 3] += sh
    ref = rng.normal(size=(N, C)) * 0.3
    poses = np.zeros((n_hyp, 12), np.float32)
    for m in range(n_hyp):
        Tm = T.copy()
        if m > 0:
            Tm[:, :3] = T[:, :3] @ Rotation.from_rotvec(rng.normal(size=3) * 0.01).as_matrix()
            Tm[:, 3] += rng.normal(size=3) * 0.3
        poses[m] = Tm.reshape(-1)
    enc = (lambda a: np.ascontiguousarray(a, np.float32))
    if dtype == "bf16":
        from paper_2606_31098_b200.workloads import to_bf16_bits
        enc = to_bf16_bits
    elif dtype == "f16":
        enc = (lambda a: np.ascontiguousarray(a, np.float16))
    g = np.array([0.05, -0.02, -1.0]); g /= np.linalg.norm(g)
    prob = dict(name="tiny", n_levels=1, dtype=dtype, width=[W], height=[H], channels=[C],
                query_feat=[enc(F.astype(np.float32))],
                query_conf=[rng.uniform(0.2, 1.0, (H, W)).astype(np.float32) if conf else None],
                intrinsics=[K], points=[P.astype(np.float32)], ref_feat=[enc(ref.astype(np.float32))],
                init_poses=poses, gravity_world=np.array([0.0, 0.0, -1.0]), gravity_imu=T[:, :3].T @ g,
                range_ray_cam=np.array([0.0, 0.0, 1.0]), range_meas=80.0,
                dsm=dsm.astype(np.float32), dsm_origin=(origin[0] + sh[0], origin[1] + sh[1]), dsm_gsd=gsd,
                params=dict(iters=[3], loss="l2", min_valid=1), gt_pose=T.reshape(-1), affine=aff, K=K)
    if dsm_plane is not None and sh[2] != 0.0:
        prob["dsm"] = (dsm + sh[2]).astype(np.float32)
    elif sh[2] != 0.0:
        prob["dsm"] = (dsm + sh[2]).astype(np.float32)
    return prob

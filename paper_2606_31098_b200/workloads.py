"""Seeded synthetic workloads for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (tests, cpu_baseline) and the CUDA path with the
same input bytes. It holds none of the refinement method's arithmetic: scenes are built
from analytic fields (closed-form evaluation, never bilinear interpolation), library
routines (scipy Rotation, scipy.ndimage.map_coordinates) and a pinhole camera used only to
place the scene. It imports neither the oracle nor the CUDA binding.

A problem is a plain dict of numpy host arrays:
  n_levels, width[l], height[l], channels[l], dtype ("f32"|"bf16"|"f16"),
  query_feat[l]   [H_l, W_l, C] float32 (f32) / uint16 bit patterns (bf16) / float16 (f16)
  query_conf[l]   None or [H_l, W_l] float32
  intrinsics[l]   (fx, fy, cx, cy)
  points[l]       [N, 4] float32 = x, y, z, w_ref       (geo-anchors)
  ref_feat[l]     [N, C] same element type as query_feat
  init_poses      [H, 12] float32 row-major [R_wc | C]  (pose hypotheses)
  gravity_world, gravity_imu, range_ray_cam (3,), range_meas
  dsm [Hd, Wd] float32, dsm_origin (ox, oy), dsm_gsd
  params          dict of LM parameters (names of include/pilot_refine.h)
  gt_pose         [12] float64, name, units (= sum_l H*N_l*K_l)

The paper measured on SynthCity-6 / UAVScenes / UAVD4L-2yr with trained descriptors
(PAPER.md:180-193); none of that is reproducible here. These inputs stand in for it with the
paper's shapes: 3-level pyramid of 32-ch descriptors, hundreds to thousands of
anchors, 10^2-10^3 hypotheses, oblique views.
"""
import copy
from concurrent.futures import ThreadPoolExecutor

import numpy as np
from scipy.ndimage import map_coordinates
from scipy.spatial.transform import Rotation

BASE_SEED = 20260631


# ------------------------------------------------------------------ element types

def to_bf16_bits(a):
    """float32 -> bf16 bit patterns (uint16), round to nearest even."""
    u = np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)
    r = ((u >> 16) & 1) + np.uint32(0x7FFF)
    return ((u + r) >> 16).astype(np.uint16)


def bf16_bits_to_f32(b):
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32)


def encode(a, dtype):
    if dtype == "f32":
        return np.ascontiguousarray(a, dtype=np.float32)
    if dtype == "bf16":
        return to_bf16_bits(a)
    if dtype == "f16":
        return np.ascontiguousarray(a, dtype=np.float16)
    raise ValueError(dtype)


def decode(a, dtype):
    if dtype == "bf16":
        return bf16_bits_to_f32(a)
    return np.asarray(a, dtype=np.float32)


# ------------------------------------------------------------------ analytic fields

class GaussianField:
    """channel c = sum_k a_kc exp(-|x - mu_kc|^2 / (2 s_kc^2)), coordinates in pixels (config 0)."""

    def __init__(self, rng, C, n_comp, W, H, sig_lo, sig_hi):
        self.a = rng.uniform(-1, 1, (n_comp, C))
        self.mx = rng.uniform(0, W - 1, (n_comp, C))
        self.my = rng.uniform(0, H - 1, (n_comp, C))
        self.s = rng.uniform(sig_lo, sig_hi, (n_comp, C))

    def at(self, x, y, n_comp=None):
        """x, y: arrays [...]; returns [..., C] float64."""
        x = np.asarray(x, np.float64)[..., None, None]
        y = np.asarray(y, np.float64)[..., None, None]
        e = np.exp(-((x - self.mx) ** 2 + (y - self.my) ** 2) / (2 * self.s ** 2))
        return (self.a * e).sum(-2)


class SinusoidField:
    """channel c = sum_{k<K} a_kc/sqrt(K) sin(2 pi (x cos t_kc + y sin t_kc)/L_kc + p_kc), x,y in FINE pixels."""

    def __init__(self, rng, C, bands, per_band):
        lam = [np.exp(rng.uniform(np.log(lo), np.log(hi), (per_band, C))) for lo, hi in bands]
        self.lam = np.concatenate(lam, 0)                      # lowest-frequency band first
        n = self.lam.shape[0]
        self.th = rng.uniform(0, 2 * np.pi, (n, C))
        self.ph = rng.uniform(0, 2 * np.pi, (n, C))
        self.a = rng.uniform(0.5, 1.0, (n, C))
        self.kx = 2 * np.pi * np.cos(self.th) / self.lam
        self.ky = 2 * np.pi * np.sin(self.th) / self.lam

    def at(self, x, y, n_comp):
        x = np.asarray(x, np.float64)[..., None, None]
        y = np.asarray(y, np.float64)[..., None, None]
        K = n_comp
        v = self.a[:K] * np.sin(self.kx[:K] * x + self.ky[:K] * y + self.ph[:K])
        return v.sum(-2) / np.sqrt(K)

    def grid(self, W, H, scale, n_comp):
        """Field at level pixels (x, y) <-> fine coords (x/scale, y/scale); separable evaluation. [H, W, C] f32."""
        K = n_comp
        xs = (np.arange(W, dtype=np.float64) / scale)[:, None, None]
        ys = (np.arange(H, dtype=np.float64) / scale)[:, None, None]
        ax = self.kx[:K] * xs + self.ph[:K]                    # [W, K, C]
        ay = self.ky[:K] * ys                                  # [H, K, C]
        amp = self.a[:K] / np.sqrt(K)
        sx, cx = (amp * np.sin(ax)).astype(np.float32), (amp * np.cos(ax)).astype(np.float32)
        sy, cy = np.sin(ay).astype(np.float32), np.cos(ay).astype(np.float32)
        # sin(A + B) = sin A cos B + cos A sin B, summed over k
        out = np.einsum("xkc,ykc->yxc", sx, cy, optimize=True) + np.einsum("xkc,ykc->yxc", cx, sy, optimize=True)
        return np.ascontiguousarray(out, dtype=np.float32)


# ------------------------------------------------------------------ heightfields

def gaussian_dsm(rng, n, size, n_bumps, amp_lo, amp_hi, sig_lo, sig_hi, mode):
    """size x size heightfield of Gaussian bumps (sigma in samples): mode 'sum' or 'max'."""
    ys, xs = np.mgrid[0:size, 0:size].astype(np.float32)
    z = np.zeros((size, size), np.float32)
    for _ in range(n_bumps):
        a = rng.uniform(amp_lo, amp_hi)
        s = rng.uniform(sig_lo, sig_hi)
        mx, my = rng.uniform(0, size - 1, 2)
        r = int(4 * s) + 1
        x0, x1 = max(0, int(mx) - r), min(size, int(mx) + r + 1)
        y0, y1 = max(0, int(my) - r), min(size, int(my) + r + 1)
        b = (a * np.exp(-((xs[y0:y1, x0:x1] - mx) ** 2 + (ys[y0:y1, x0:x1] - my) ** 2) / (2 * s * s))).astype(np.float32)
        if mode == "sum":
            z[y0:y1, x0:x1] += b
        else:
            z[y0:y1, x0:x1] = np.maximum(z[y0:y1, x0:x1], b)
    return z


def dsm_height(dsm, origin, gsd, x, y):
    """Height under world (x, y) by the library's order-1 spline (scene placement only)."""
    gx = (np.asarray(x, np.float64) - origin[0]) / gsd
    gy = (np.asarray(y, np.float64) - origin[1]) / gsd
    return map_coordinates(dsm.astype(np.float64), [np.atleast_1d(gy), np.atleast_1d(gx)], order=1, mode="nearest")


# ------------------------------------------------------------------ camera placement

def look_pose(C, forward):
    """[R_wc | C] with camera x right, y down, z forward; world z up."""
    f = np.asarray(forward, np.float64)
    f = f / np.linalg.norm(f)
    right = np.cross(f, [0.0, 0.0, 1.0])
    right /= np.linalg.norm(right)
    down = np.cross(f, right)
    T = np.zeros((3, 4))
    T[:, 0], T[:, 1], T[:, 2], T[:, 3] = right, down, f, C
    return T


def pitched_pose(C, pitch_deg, heading_deg=0.0):
    """Optical axis pitch_deg below horizontal; heading 0 = +y, positive towards +x."""
    p, h = np.deg2rad(pitch_deg), np.deg2rad(heading_deg)
    return look_pose(C, [np.cos(p) * np.sin(h), np.cos(p) * np.cos(h), -np.sin(p)])


def project(T, K, P):
    """Pinhole placement of world points P [N,3] through pose T=[R_wc|C], K=(fx,fy,cx,cy): (u, v, Z)."""
    pc = (P - T[:, 3]) @ T[:, :3]
    return K[0] * pc[:, 0] / pc[:, 2] + K[2], K[1] * pc[:, 1] / pc[:, 2] + K[3], pc[:, 2]


def perturbed_poses(rng, T_gt, H, rot_deg, trans_m, first_is_gt, fixed_norm=False):
    """R_wc_m = R_wc_gt Rot(d), C_m = C_gt + t. Per-axis uniform (or fixed magnitude, random direction)."""
    out = np.zeros((H, 12), np.float32)
    for m in range(H):
        if fixed_norm:
            d = rng.normal(size=3); d *= np.deg2rad(rot_deg) / np.linalg.norm(d)
            t = rng.normal(size=3); t *= trans_m / np.linalg.norm(t)
        else:
            d = np.deg2rad(rng.uniform(-rot_deg, rot_deg, 3))
            t = rng.uniform(-trans_m, trans_m, 3)
        if first_is_gt and m == 0:
            d, t = np.zeros(3), np.zeros(3)
        T = np.zeros((3, 4))
        T[:, :3] = T_gt[:, :3] @ Rotation.from_rotvec(d).as_matrix()
        T[:, 3] = T_gt[:, 3] + t
        out[m] = T.reshape(-1).astype(np.float32)
    return out


def morton_order(ix, iy):
    """Permutation sorting integer grid nodes by Morton (Z-order) code: spatially coherent point order."""
    def spread(v):
        v = v.astype(np.uint64) & np.uint64(0xFFFF)
        v = (v | (v << np.uint64(8))) & np.uint64(0x00FF00FF)
        v = (v | (v << np.uint64(4))) & np.uint64(0x0F0F0F0F)
        v = (v | (v << np.uint64(2))) & np.uint64(0x33333333)
        v = (v | (v << np.uint64(1))) & np.uint64(0x55555555)
        return v
    return np.argsort(spread(ix) | (spread(iy) << np.uint64(1)), kind="stable")


def centre_range(dsm, origin, gsd, T, v_cam, t_max):
    """Distance along the centre ray to the heightfield: dense sampling + linear refinement (measurement synthesis)."""
    w = T[:, :3] @ np.asarray(v_cam, np.float64)
    t = np.linspace(0.0, t_max, 20001)
    P = T[:, 3][None, :] + t[:, None] * w[None, :]
    f = P[:, 2] - dsm_height(dsm, origin, gsd, P[:, 0], P[:, 1])
    idx = np.nonzero((f[:-1] > 0) & (f[1:] <= 0))[0]
    if idx.size == 0:
        return float("nan")
    i = idx[0]
    return float(t[i] + (t[i + 1] - t[i]) * f[i] / (f[i] - f[i + 1]))


# ------------------------------------------------------------------ scene assembly

def _grid_points(rng, dsm, origin, gsd, N, region=None):
    """N geo-anchors at random DSM grid nodes (z = the node's height, no interpolation), Morton-sorted."""
    Hd, Wd = dsm.shape
    if region is None:
        x0, x1, y0, y1 = 1, Wd - 1, 1, Hd - 1
    else:
        x0, x1, y0, y1 = region
    ix = rng.integers(x0, x1, N)
    iy = rng.integers(y0, y1, N)
    o = morton_order(ix - x0, iy - y0)
    ix, iy = ix[o], iy[o]
    P = np.stack([origin[0] + ix * gsd, origin[1] + iy * gsd, dsm[iy, ix].astype(np.float64)], 1)
    return P


def _assemble(name, rng, field, levels, dtype, P, T_gt, K_fine, noise, dsm, origin, gsd, poses, params,
              n_comp, gauss_level_scale=None):
    """levels: list of (W, H, C, scale). Builds maps, reference features (analytic field at the GT projection + noise)."""
    prob = dict(name=name, n_levels=len(levels), dtype=dtype, width=[], height=[], channels=[],
                query_feat=[], query_conf=[], intrinsics=[], points=[], ref_feat=[])
    u, v, _ = project(T_gt, K_fine, P)                       # fine-level pixel coordinates of every anchor at GT
    pts = np.concatenate([P, np.ones((P.shape[0], 1))], 1).astype(np.float32)
    for li, (W, H, C, s) in enumerate(levels):
        K = n_comp[li]
        if isinstance(field, SinusoidField):
            grid = field.grid(W, H, s, K)
        else:
            ys, xs = np.mgrid[0:H, 0:W]
            grid = field.at(xs / s, ys / s).astype(np.float32)
        ref = np.concatenate([field.at(u[i:i + 4096], v[i:i + 4096], K) for i in range(0, P.shape[0], 4096)], 0) \
            if P.shape[0] else np.zeros((0, C))
        ref = ref + rng.normal(0.0, noise, ref.shape)
        prob["width"].append(W); prob["height"].append(H); prob["channels"].append(C)
        prob["query_feat"].append(encode(grid, dtype))
        prob["query_conf"].append(None)
        prob["intrinsics"].append(tuple(float(k * s) for k in K_fine))
        prob["points"].append(pts)
        prob["ref_feat"].append(encode(ref.astype(np.float32), dtype))
    prob.update(init_poses=poses, dsm=dsm, dsm_origin=(float(origin[0]), float(origin[1])), dsm_gsd=float(gsd),
                gravity_world=np.array([0.0, 0.0, -1.0]), gravity_imu=np.array([0.0, 0.0, -1.0]),
                range_ray_cam=np.array([0.0, 0.0, 1.0]), range_meas=1.0, params=params,
                gt_pose=T_gt.reshape(-1).copy())
    prob["units"] = int(sum(poses.shape[0] * P.shape[0] * k for k in params["iters"]))
    return prob


def _sensors(prob, rng, T_gt, tilt_sigma_deg, range_sigma, t_max):
    """gamma^imu = R_cw,GT gamma^W tilted by N(0, sigma); d_meas = centre-ray range from GT + N(0, sigma)."""
    e = T_gt[:, :3].T @ prob["gravity_world"]
    tilt = Rotation.from_rotvec(np.deg2rad(rng.normal(0.0, tilt_sigma_deg, 3))).as_matrix()
    g = tilt @ e
    prob["gravity_imu"] = g / np.linalg.norm(g)
    d = centre_range(prob["dsm"], prob["dsm_origin"], prob["dsm_gsd"], T_gt, prob["range_ray_cam"], t_max)
    prob["range_meas"] = float(d + rng.normal(0.0, range_sigma))
    prob["range_true"] = d


def _rng(idx):
    return np.random.Generator(np.random.PCG64(BASE_SEED + idx))


def config0(noise=0.01):
    """Tiny CPU-seconds case (BASELINE.json configs[0])."""
    rng = _rng(0)
    W, H, C = 64, 48, 16
    field = GaussianField(rng, C, 8, W, H, 4.0, 12.0)
    dsm = gaussian_dsm(rng, 0, 64, 5, 0.0, 4.0, 6.0, 16.0, "sum")
    gsd, origin = 1.0, (-31.5, -31.5)
    P = _grid_points(rng, dsm, origin, gsd, 256)
    h0 = float(dsm_height(dsm, origin, gsd, 0.0, 0.0)[0])
    T_gt = pitched_pose([0.0, -100.0, h0 + 100.0], 45.0)
    poses = perturbed_poses(rng, T_gt, 1, 2.0, 2.0, first_is_gt=False, fixed_norm=True)
    params = dict(iters=[5], loss="cauchy", loss_scale=0.1, w_gravity=0.0, range_mode="off", min_valid=16)
    return _assemble("config0", rng, field, [(W, H, C, 1.0)], "f32", P, T_gt, (60.0, 60.0, 32.0, 24.0), noise,
                     dsm, origin, gsd, poses, params, [8])


def _pilot_scene(rng, dsm_size, gsd, n_bumps, fine_w, fine_h):
    dsm = gaussian_dsm(rng, 0, dsm_size, n_bumps, 5.0, 40.0, 8.0, 30.0, "max")
    ext = dsm_size * gsd
    origin = (-(dsm_size - 1) * gsd / 2, -(dsm_size - 1) * gsd / 2)
    alt = 0.6 * ext
    zc = float(dsm.mean())
    C = np.array([0.0, -alt, zc + alt])
    T_gt = look_pose(C, np.array([0.0, 0.0, zc]) - C)        # 45 deg, aimed at the crop centre
    f = fine_w / 2 / np.tan(np.deg2rad(31.0))
    return dsm, origin, ext, T_gt, (f, f, fine_w / 2.0, fine_h / 2.0)


BANDS = [(128.0, 512.0), (48.0, 128.0), (16.0, 48.0)]        # fine-pixel wavelengths, 4 components each


def config1(H=64, N=4096, iters=(10, 10, 10), idx=1):
    """PiLoT-like frame (BASELINE.json configs[1])."""
    rng = _rng(idx)
    field = SinusoidField(rng, 32, BANDS, 4)
    dsm, origin, ext, T_gt, K = _pilot_scene(rng, 512, 0.5, 40, 480, 270)
    P = _grid_points(rng, dsm, origin, 0.5, N)
    poses = perturbed_poses(rng, T_gt, H, 5.0, 10.0, first_is_gt=True)
    params = dict(iters=list(iters), loss="huber", loss_scale=0.1, w_gravity=1.0, gravity_scale=0.1,
                  range_mode="march", w_range=1.0, range_scale=5.0, min_valid=max(8, N // 16))
    levels = [(120, 68, 32, 0.25), (240, 135, 32, 0.5), (480, 270, 32, 1.0)]
    prob = _assemble("config1", rng, field, levels, "bf16", P, T_gt, K, 0.02, dsm, origin, 0.5, poses, params,
                     [4, 8, 12])
    _sensors(prob, rng, T_gt, 0.1, 0.5, 4 * ext)
    return prob


def config2(H=1024, N=8192, iters=20):
    """Hypothesis-throughput stress (BASELINE.json configs[2]); low band only so +-10 deg stays in the basin."""
    rng = _rng(2)
    field = SinusoidField(rng, 64, BANDS[:1], 4)
    dsm, origin, ext, T_gt, K = _pilot_scene(rng, 512, 0.5, 40, 480, 270)
    P = _grid_points(rng, dsm, origin, 0.5, N)
    poses = perturbed_poses(rng, T_gt, H, 10.0, 20.0, first_is_gt=True)
    params = dict(iters=[iters], loss="huber", loss_scale=0.1, w_gravity=1.0, gravity_scale=0.1,
                  range_mode="march", w_range=1.0, range_scale=5.0, min_valid=max(8, N // 16))
    prob = _assemble("config2", rng, field, [(480, 270, 64, 1.0)], "bf16", P, T_gt, K, 0.02, dsm, origin, 0.5,
                     poses, params, [4])
    _sensors(prob, rng, T_gt, 0.1, 0.5, 4 * ext)
    return prob


def config4(H=256, N=65536, iters=10, width=1920, height=1080, dsm_size=4096):
    """High-resolution, L2-exceeding case (BASELINE.json configs[4]): 265 MB map, HBM-side gather."""
    rng = _rng(4)
    field = SinusoidField(rng, 64, [(512.0, 2048.0)], 4)
    gsd = 0.25 * 4096 / dsm_size
    dsm, origin, ext, T_gt, K = _pilot_scene(rng, dsm_size, gsd, 40 * (dsm_size // 512) ** 2 // 4, width, height)
    P = _grid_points(rng, dsm, origin, gsd, N)
    poses = perturbed_poses(rng, T_gt, H, 5.0, 10.0, first_is_gt=True)
    params = dict(iters=[iters], loss="cauchy", loss_scale=0.1, w_gravity=1.0, gravity_scale=0.1,
                  range_mode="march", w_range=1.0, range_scale=5.0, min_valid=max(8, N // 16))
    prob = _assemble("config4", rng, field, [(width, height, 64, 1.0)], "bf16", P, T_gt, K, 0.02, dsm, origin, gsd,
                     poses, params, [4])
    _sensors(prob, rng, T_gt, 0.1, 0.5, 4 * ext)
    return prob


# ------------------------------------------------------------------ config 3: streaming sequence

def _normalize(v):
    v = np.asarray(v, np.float64)
    return v / np.linalg.norm(v)


class Config3Sequence:
    """Streaming sequence (BASELINE.json configs[3]): `n_frames` frames along a circular trajectory over one
    2048x2048 heightfield @ 0.5 m; frames are generated lazily (`frame(i)`), each a problem dict WITHOUT init_poses
    (the harness seeds them from the previous frame's estimate: `offsets` is the fixed table of +-5 deg / +-10 m
    camera-frame offsets, entry 0 = identity; "pose estimated from the previous query image ... as the
    pose prior"). Radius 300 m, 15 m/s at 30 fps, 150 m above the mean terrain, heading tangent, pitch
    45 + 15 sin(2 pi i / 300) deg (30-60 deg oblique)."""

    LEVELS = [(120, 68, 32, 0.25), (240, 135, 32, 0.5), (480, 270, 32, 1.0)]

    def __init__(self, n_frames=300, H=128, N=4096, iters=(10, 10, 10), dsm_size=2048):
        rng = _rng(3)
        self.n_frames, self.H, self.N, self.iters = n_frames, H, N, list(iters)
        self.gsd = 0.5
        self.dsm = gaussian_dsm(rng, 0, dsm_size, 40 * (dsm_size // 512) ** 2, 5.0, 40.0, 8.0, 30.0, "max")
        self.dsm64 = self.dsm.astype(np.float64)
        self.origin = (-(dsm_size - 1) * self.gsd / 2, -(dsm_size - 1) * self.gsd / 2)
        self.z_mean = float(self.dsm.mean())
        self.field = SinusoidField(rng, 32, BANDS, 4)
        self.dph = rng.uniform(-0.05, 0.05, self.field.ph.shape)           # phase drift per frame (rad)
        self.ph0 = self.field.ph.copy()
        f = 480 / 2 / np.tan(np.deg2rad(31.0))
        self.K = (f, f, 240.0, 135.0)
        off = np.zeros((H, 6), np.float32)
        off[:, :3] = np.deg2rad(rng.uniform(-5.0, 5.0, (H, 3)))
        off[:, 3:] = rng.uniform(-10.0, 10.0, (H, 3))
        off[0] = 0
        self.offsets = off
        self.params = dict(iters=list(iters), loss="huber", loss_scale=0.1, w_gravity=1.0, gravity_scale=0.1,
                           range_mode="march", w_range=1.0, range_scale=5.0, min_valid=max(8, N // 16))
        self.gravity_world = np.array([0.0, 0.0, -1.0])
        self.units_per_frame = int(sum(H * N * k for k in iters))

    def gt_pose(self, i):
        phi = 0.5 * i / 300.0                                             # 0.5 m per frame on a 300 m circle
        C = np.array([300.0 * np.cos(phi), 300.0 * np.sin(phi), self.z_mean + 150.0])
        pitch = 45.0 + 15.0 * np.sin(2 * np.pi * i / 300.0)
        return pitched_pose(C, pitch, np.rad2deg(-phi))                   # heading tangent to the circle

    def _height(self, x, y):
        gx = (np.asarray(x, np.float64) - self.origin[0]) / self.gsd
        gy = (np.asarray(y, np.float64) - self.origin[1]) / self.gsd
        return map_coordinates(self.dsm64, [np.atleast_1d(gy), np.atleast_1d(gx)], order=1, mode="nearest")

    def frame(self, i):
        rng = np.random.Generator(np.random.PCG64([BASE_SEED + 3, i + 1]))
        T = self.gt_pose(i)
        # anchors: DSM nodes in a 256 m square centred on the ground point under the optical axis
        fwd = T[:, 2]
        t = (T[2, 3] - self.z_mean) / -fwd[2]
        gx = (T[0, 3] + t * fwd[0] - self.origin[0]) / self.gsd
        gy = (T[1, 3] + t * fwd[1] - self.origin[1]) / self.gsd
        half = int(128 / self.gsd)
        Hd, Wd = self.dsm.shape
        region = (max(1, int(gx) - half), min(Wd - 1, int(gx) + half), max(1, int(gy) - half), min(Hd - 1, int(gy) + half))
        P = _grid_points(rng, self.dsm, self.origin, self.gsd, self.N, region)
        field = copy.copy(self.field)                                     # thread-safe: frames may be built in parallel
        field.ph = self.ph0 + i * self.dph
        prob = _assemble("config3", rng, field, self.LEVELS, "bf16", P, T, self.K, 0.02, self.dsm, self.origin,
                         self.gsd, np.zeros((0, 12), np.float32), dict(self.params), [4, 8, 12])
        prob.pop("init_poses")
        prob["units"] = self.units_per_frame
        prob["frame"] = i
        # sensors (as _sensors, with the cached float64 heightfield)
        e = T[:, :3].T @ self.gravity_world
        tilt = Rotation.from_rotvec(np.deg2rad(rng.normal(0.0, 0.1, 3))).as_matrix()
        prob["gravity_imu"] = _normalize(tilt @ e)
        w = T[:, :3] @ prob["range_ray_cam"]
        ts = np.linspace(0.0, 2000.0, 20001)
        Pr = T[:, 3][None, :] + ts[:, None] * w[None, :]
        fz = Pr[:, 2] - self._height(Pr[:, 0], Pr[:, 1])
        k = np.nonzero((fz[:-1] > 0) & (fz[1:] <= 0))[0][0]
        d = float(ts[k] + (ts[k + 1] - ts[k]) * fz[k] / (fz[k] - fz[k + 1]))
        prob["range_true"] = d
        prob["range_meas"] = float(d + rng.normal(0.0, 0.5))
        return prob


    def frames(self, indices=None, workers=8, ahead=16):
        """Generator over frame dicts, built `ahead` frames in advance on a thread pool (numpy releases the GIL)."""
        idx = list(range(self.n_frames) if indices is None else indices)
        with ThreadPoolExecutor(max_workers=workers) as ex:
            pending = [ex.submit(self.frame, i) for i in idx[:ahead]]
            nxt = len(pending)
            while pending:
                fut = pending.pop(0)
                if nxt < len(idx):
                    pending.append(ex.submit(self.frame, idx[nxt]))
                    nxt += 1
                yield fut.result()


def with_poses(frame_prob, poses):
    """A frame of Config3Sequence / paper_frame plus a hypothesis set -> a complete problem dict."""
    q = dict(frame_prob)
    q["init_poses"] = np.ascontiguousarray(poses, np.float32).reshape(-1, 12)
    return q


# ------------------------------------------------------------------ paper-shaped frame

PAPER_YAWS = (-9.0, -7.0, -5.0, -3.0, -1.0, 1.0, 3.0, 5.0, 7.0, 9.0)      # supp Eq.(4)


def paper_frame(N=500, iters=(2, 3, 4), dtype="bf16", prior_error=(3.1, -4.3, 2.2), range_mode="height"):
    """The paper's own problem shape: images resized to 512, 3-level pyramid of
    L2-normalised 32-channel descriptors with query confidence maps and per-anchor reference confidences, 500
    geo-anchors, 2/3/4 LM iterations, 1210 (x, y, psi) hypotheses around a pose prior (to be sampled by the caller
    from `prior_pose` with `grid = (10 m, 2 m, PAPER_YAWS)` in the world frame), top 128 kept after the coarse level.
    Stand-in for the paper's data: analytic sinusoid descriptors, Gaussian-building DSM crop.
    prior_error = (dx m, dy m, dyaw deg) of the prior w.r.t. the ground truth."""
    rng = _rng(5)
    field = SinusoidField(rng, 32, BANDS, 4)
    dsm, origin, ext, T_gt, K = _pilot_scene(rng, 512, 0.5, 40, 512, 512)
    P = _grid_points(rng, dsm, origin, 0.5, N)
    params = dict(iters=list(iters), loss="huber", loss_scale=0.1, w_gravity=1.0, gravity_scale=0.1,
                  range_mode=range_mode, w_range=1.0, range_scale=5.0, min_valid=max(8, N // 16))
    levels = [(128, 128, 32, 0.25), (256, 256, 32, 0.5), (512, 512, 32, 1.0)]
    prob = _assemble("paper_frame", rng, field, levels, "f32", P, T_gt, K, 0.02, dsm, origin, 0.5,
                     np.zeros((0, 12), np.float32), params, [4, 8, 12])
    prob.pop("init_poses")
    # channel-wise L2 normalisation of query and reference descriptors, then the storage dtype
    for l in range(3):
        q = prob["query_feat"][l].astype(np.float64)
        prob["query_feat"][l] = encode((q / np.linalg.norm(q, axis=-1, keepdims=True)).astype(np.float32), dtype)
        r = prob["ref_feat"][l].astype(np.float64)
        prob["ref_feat"][l] = encode((r / np.linalg.norm(r, axis=-1, keepdims=True)).astype(np.float32), dtype)
        W, H = prob["width"][l], prob["height"][l]
        ys, xs = np.mgrid[0:H, 0:W] / levels[l][3]
        conf = 1.0 / (1.0 + np.exp(-(1.0 + 1.5 * np.sin(xs / 70.0 + 0.3) * np.cos(ys / 55.0 - 0.2))))   # sigmoid head
        prob["query_conf"][l] = conf.astype(np.float32)
    prob["dtype"] = dtype
    w_ref = rng.uniform(0.5, 1.0, N).astype(np.float32)
    pts = prob["points"][0].copy()
    pts[:, 3] = w_ref
    prob["points"] = [pts, pts, pts]
    _sensors(prob, rng, T_gt, 0.1, 0.5, 4 * ext)
    dx, dy, dyaw = prior_error
    Tp = T_gt.copy()
    Tp[:, :3] = Rotation.from_rotvec([0.0, 0.0, np.deg2rad(dyaw)]).as_matrix() @ T_gt[:, :3]
    Tp[:, 3] = T_gt[:, 3] + [dx, dy, 0.0]
    prob["prior_pose"] = Tp.reshape(-1).astype(np.float32)
    prob["grid"] = (10.0, 2.0, PAPER_YAWS)
    prob["keep"] = 128
    H0 = 121 * len(PAPER_YAWS)
    prob["units"] = int(N * (H0 * iters[0] + prob["keep"] * (iters[1] + iters[2])))
    return prob


def make(name, **kw):
    return {"config0": config0, "config1": config1, "config2": config2, "config4": config4}[name](**kw)


def levels_slice(prob, begin, end, poses=None):
    """Sub-problem made of pyramid levels [begin, end) of `prob` (what pilot_refine_run_levels works on), optionally with
    other initial poses. Dict slicing only."""
    q = dict(prob)
    q["n_levels"] = end - begin
    for k in ("width", "height", "channels", "query_feat", "intrinsics", "points", "ref_feat"):
        q[k] = list(prob[k][begin:end])
    q["query_conf"] = list(prob.get("query_conf", [None] * prob["n_levels"])[begin:end])
    if poses is not None:
        q["init_poses"] = np.ascontiguousarray(poses, np.float32).reshape(-1, 12)
    P = dict(prob.get("params", {}))
    P["iters"] = list(P["iters"][begin:end])
    q["params"] = P
    return q

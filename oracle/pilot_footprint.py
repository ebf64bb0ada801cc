"""CPU ORACLE of the reference-crop geometry that feeds the refinement with geo-anchors (numpy, float64).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module. It shares no code with paper_2606_31098_b200/csrc.

Passages followed (arxiv/paper_2606_31098, supp II-B, PAPER.md line numbers):
  * map-footprint estimation: rays from the camera centre through the four image corners; along each ray the
    sample most consistent with the DSM surface, s* = argmin_s |z_ray(s) - h_DSM(x_ray(s), y_ray(s))|  (supp Eq.2,
    PAPER.md:363-368); the four surface points define a quadrilateral footprint
  * pixel-aligned reference warping: ONE homography maps the rectangular crop onto that quadrilateral for every
    map layer
  * geo-anchor construction: P(u, v) = [x^m(u, v), y^m(u, v), D^r(u, v)]                     (supp Eq.3)
Readings where the paper is silent (A20-A22): the search of Eq.2 is over n uniform samples
s_i = i * s_max / n, i = 1..n, samples outside the DSM are skipped, ties go to the smallest s; the warped DSM
layer D^r is the bilinear sample of the DSM at the warped map coordinates; crop pixel (0,0), (Wc-1,0), (Wc-1,Hc-1),
(0,Hc-1) correspond to the image corners (0,0), (W-1,0), (W-1,H-1), (0,H-1) in this order.

Pins (tests/test_oracle_footprint.py): closed-form ray/plane intersection on a planar DSM (the arg-min sample is
the one nearest to the analytic s); the homography reproduces its four defining correspondences, preserves
collinearity, reduces to the affine map for a parallelogram, and — over a planar DSM — the lifted anchor of crop
pixel (u, v) equals the analytic back-projection of the corresponding image pixel onto the plane (the image-to-
ground map of a pinhole camera over a plane IS a homography).
"""
import numpy as np


def dsm_bilinear(dsm, origin, gsd, x, y):
    """Bilinear heightfield sample, the rule of the refinement's range prior (in bounds iff the 2x2 cell exists)."""
    gx, gy = (x - origin[0]) / gsd, (y - origin[1]) / gsd
    ix, iy = np.floor(gx), np.floor(gy)
    Hd, Wd = dsm.shape
    if not (np.isfinite(gx) and np.isfinite(gy)) or ix < 0 or iy < 0 or ix > Wd - 2 or iy > Hd - 2:
        return None
    ix, iy = int(ix), int(iy)
    a, b = gx - ix, gy - iy
    d = dsm.astype(np.float64)
    return (1 - b) * ((1 - a) * d[iy, ix] + a * d[iy, ix + 1]) + b * ((1 - a) * d[iy + 1, ix] + a * d[iy + 1, ix + 1])


def corner_rays(pose, K, width, height):
    """World-frame unit rays through the image corners (0,0), (W-1,0), (W-1,H-1), (0,H-1); pose = [R_wc | C]."""
    T = np.asarray(pose, np.float64).reshape(3, 4)
    fx, fy, cx, cy = [float(k) for k in K]
    rays = []
    for (u, v) in [(0, 0), (width - 1, 0), (width - 1, height - 1), (0, height - 1)]:
        d = np.array([(u - cx) / fx, (v - cy) / fy, 1.0])
        d /= np.linalg.norm(d)
        rays.append(T[:, :3] @ d)
    return T[:, 3].copy(), np.asarray(rays)


def footprint(pose, K, width, height, dsm, origin, gsd, n_samples, s_max):
    """supp Eq.(2). Returns [4, 4]: x, y, z_ray at s*, and the residual |z_ray - h_DSM| there (NaN row: no sample
    of that ray lies over the DSM)."""
    C, rays = corner_rays(pose, K, width, height)
    out = np.full((4, 4), np.nan)
    for c in range(4):
        best = None
        for i in range(1, n_samples + 1):
            s = i * s_max / n_samples
            p = C + s * rays[c]
            h = dsm_bilinear(dsm, origin, gsd, p[0], p[1])
            if h is None:
                continue
            res = abs(p[2] - h)
            if best is None or res < best[0]:
                best = (res, p)
        if best is not None:
            out[c, :3], out[c, 3] = best[1], best[0]
    return out


def homography(quad_xy, crop_w, crop_h):
    """3x3 H with H (u, v, 1)^T ~ (x, y, 1)^T for the four crop corners -> quad_xy [4, 2] (library linear solve)."""
    src = [(0.0, 0.0), (crop_w - 1.0, 0.0), (crop_w - 1.0, crop_h - 1.0), (0.0, crop_h - 1.0)]
    A, b = np.zeros((8, 8)), np.zeros(8)
    for k, ((u, v), (x, y)) in enumerate(zip(src, np.asarray(quad_xy, np.float64))):
        A[2 * k] = [u, v, 1, 0, 0, 0, -u * x, -v * x]
        A[2 * k + 1] = [0, 0, 0, u, v, 1, -u * y, -v * y]
        b[2 * k], b[2 * k + 1] = x, y
    h = np.linalg.solve(A, b)
    return np.append(h, 1.0).reshape(3, 3)


def lift_anchors(corners, crop_w, crop_h, pix, dsm, origin, gsd):
    """supp Eq.(3): crop pixels pix [N, 2] -> anchors [N, 4] = x^m, y^m, D^r, w (w = 1 valid, 0 = outside the DSM,
    in which case z = 0)."""
    Hm = homography(np.asarray(corners, np.float64)[:, :2], crop_w, crop_h)
    out = np.zeros((len(pix), 4))
    for k, (u, v) in enumerate(np.asarray(pix, np.float64)):
        q = Hm @ np.array([u, v, 1.0])
        x, y = q[0] / q[2], q[1] / q[2]
        h = dsm_bilinear(dsm, origin, gsd, x, y)
        out[k] = [x, y, 0.0 if h is None else h, 0.0 if h is None else 1.0]
    return out

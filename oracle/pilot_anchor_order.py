"""Oracle of the anchor ordering (include/pilot_refine.h, pilot_refine_sort_anchors).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import this module.
Plain numpy, the definition written out: bounding box of the anchors' (x, y); 16-bit quantisation
q = floor((v - min) * (65535 / (max - min))) in float32 (the decisions are integers, so both sides take them in the
kernel's precision: one IEEE float32 operation per step, which numpy float32 scalars/arrays reproduce exactly); Morton key =
bit-interleaving of q_x (even bits) and q_y (odd bits); a STABLE sort of the keys. It imports nothing from the product.
"""
import numpy as np


def quant16(v, lo, hi):
    v = np.asarray(v, np.float32)
    ext = np.float32(hi) - np.float32(lo)
    if not ext > 0:
        return np.zeros(v.shape, np.uint32)
    scale = np.float32(65535.0) / ext
    t = np.floor((v - np.float32(lo)) * scale)
    t = np.where(np.isfinite(v), t, np.float32(0))
    return np.clip(t, 0, 65535).astype(np.uint32)


def interleave16(qx, qy):
    """Bit i of qx -> bit 2i, bit i of qy -> bit 2i+1, one bit at a time (the definition, not the magic-number spread)."""
    key = np.zeros(np.shape(qx), np.uint64)
    for i in range(16):
        key |= ((np.asarray(qx, np.uint64) >> np.uint64(i)) & np.uint64(1)) << np.uint64(2 * i)
        key |= ((np.asarray(qy, np.uint64) >> np.uint64(i)) & np.uint64(1)) << np.uint64(2 * i + 1)
    return key.astype(np.uint32)


def morton_keys(points):
    P = np.asarray(points, np.float32).reshape(-1, 4)
    ok = np.isfinite(P[:, 0]) & np.isfinite(P[:, 1])
    if not ok.any():
        return np.zeros(P.shape[0], np.uint32)
    lox, loy = P[ok, 0].min(), P[ok, 1].min()
    hix, hiy = P[ok, 0].max(), P[ok, 1].max()
    return interleave16(quant16(P[:, 0], lox, hix), quant16(P[:, 1], loy, hiy))


def morton_order(points):
    """perm such that points[perm] is in Morton order; equal keys keep their input order."""
    return np.argsort(morton_keys(points), kind="stable").astype(np.int32)

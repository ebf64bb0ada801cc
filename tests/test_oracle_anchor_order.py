"""Pins of the anchor-ordering oracle (oracle/pilot_anchor_order.py): the Z-curve on small grids (textbook sequence), the
quantisation's end points, stability, and that the order is a permutation. CPU only."""
import numpy as np

from oracle import pilot_anchor_order as ao


def grid_points(nx, ny):
    ys, xs = np.mgrid[0:ny, 0:nx]
    P = np.zeros((nx * ny, 4), np.float32)
    P[:, 0], P[:, 1], P[:, 3] = xs.reshape(-1), ys.reshape(-1), 1.0
    return P


def test_z_curve_on_2x2_and_4x4_grids():
    # the Z-order (Morton) curve visits (x, y): (0,0) (1,0) (0,1) (1,1) | then the next 2x2 block to the right, ...
    P = grid_points(2, 2)
    assert [tuple(P[i, :2].astype(int)) for i in ao.morton_order(P)] == [(0, 0), (1, 0), (0, 1), (1, 1)]
    P = grid_points(4, 4)
    want = [(0, 0), (1, 0), (0, 1), (1, 1), (2, 0), (3, 0), (2, 1), (3, 1),
            (0, 2), (1, 2), (0, 3), (1, 3), (2, 2), (3, 2), (2, 3), (3, 3)]
    assert [tuple(P[i, :2].astype(int)) for i in ao.morton_order(P)] == want


def test_interleave_bit_by_bit_and_quantisation_end_points():
    assert ao.interleave16(np.array([0xffff]), np.array([0])) [0] == 0x55555555
    assert ao.interleave16(np.array([0]), np.array([0xffff]))[0] == 0xaaaaaaaa
    assert ao.interleave16(np.array([0b101]), np.array([0b011]))[0] == 0b011011       # x bits 1,0,1 on even, y bits 0,1,1 on odd
    q = ao.quant16(np.array([-3.0, 5.0, 1.0], np.float32), -3.0, 5.0)
    assert q[0] == 0 and q[1] == 65535 and q[2] == 32767
    assert np.all(ao.quant16(np.array([1.0, 2.0], np.float32), 4.0, 4.0) == 0)      # degenerate box
    assert ao.quant16(np.array([np.nan], np.float32), 0.0, 1.0)[0] == 0


def test_order_is_a_stable_permutation_and_groups_neighbours():
    rng = np.random.default_rng(3)
    P = np.zeros((5000, 4), np.float32)
    P[:, :2] = rng.uniform(-300, 300, (5000, 2))
    P[100:110, :2] = P[100, :2]                                                     # ten anchors on one spot: equal keys
    perm = ao.morton_order(P)
    assert sorted(perm.tolist()) == list(range(5000))
    pos = {int(j): k for k, j in enumerate(perm)}
    assert [pos[j] for j in range(100, 110)] == list(range(pos[100], pos[100] + 10))  # input order kept inside the tie
    # locality: consecutive anchors of the Morton order are far closer than consecutive anchors of the input order
    d_sorted = np.linalg.norm(np.diff(P[perm, :2], axis=0), axis=1).mean()
    d_input = np.linalg.norm(np.diff(P[:, :2], axis=0), axis=1).mean()
    assert d_sorted < 0.1 * d_input

"""CPU ORACLE of the hypothesis-set operations around the LM refinement (numpy, float64).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module. It shares no code with paper_2606_31098_b200/csrc.

Passages followed (arxiv/paper_2606_31098, PAPER.md line numbers):
  * sampling in the local (x, y, psi) space around the propagated pose prior
  * +-10 m grid, 2 m step, yaw offsets {+-1,+-3,+-5,+-7,+-9} deg => 1210           PAPER.md:381-386 (supp Eq.4)
  * ranking by the post-update objective after the coarse level, top 128 retained PAPER.md:386
  * the hypothesis with the lowest final objective value is the output pose
  * sequential localisation: the previous frame's estimate is the next prior
Each function is the plain definition written out; library primitives used as steps: the rotation-vector
exponential (scipy Rotation.from_rotvec), argmin, lexsort.

Pins (tests/test_oracle_hypotheses.py): 1210 = the paper's count (tests/golden/paper_counts.txt); the grid's
extreme/centre entries; Rot(w) against scipy.linalg.expm of the skew matrix; world-yaw offsets leave the
gravity residual of Eq.(3) unchanged ("yaw is not directly constrained by gravity"); camera-frame
offsets reproduce the workload generator's perturbation convention; top-k against a brute-force selection on
tiny inputs and against a full sort; argmin tie / NaN rules.
"""
import numpy as np
from scipy.spatial.transform import Rotation

SEED_CAMERA, SEED_WORLD = 0, 1


def grid_offsets(xy_range, xy_step, yaw_deg, up):
    """supp II-C: [(2r+1)^2 * n_yaw, 6] = (rotation vector rad, translation m).

    t = (i*step, j*step, 0), i, j in [-r, r]; w = radians(yaw) * up. index = ((i+r)*(2r+1) + (j+r))*n_yaw + k.
    """
    r = int(np.floor(xy_range / xy_step + 1e-6))
    up = np.asarray(up, np.float64)
    out = []
    for i in range(-r, r + 1):
        for j in range(-r, r + 1):
            for y in yaw_deg:
                w = np.deg2rad(float(y)) * up
                out.append([w[0], w[1], w[2], i * xy_step, j * xy_step, 0.0])
    return np.asarray(out, np.float64).reshape(-1, 6)


def seed_hypotheses(base_pose, offsets, frame):
    """hypotheses around a pose prior. base_pose [12] = [R_wc | C]; offsets [n, 6]. -> [n, 12]."""
    T = np.asarray(base_pose, np.float64).reshape(3, 4)
    off = np.asarray(offsets, np.float64).reshape(-1, 6)
    out = np.zeros((off.shape[0], 3, 4))
    for m in range(off.shape[0]):
        Rw = Rotation.from_rotvec(off[m, :3]).as_matrix()
        out[m, :, :3] = T[:, :3] @ Rw if frame == SEED_CAMERA else Rw @ T[:, :3]
        out[m, :, 3] = T[:, 3] + off[m, 3:]
    return out.reshape(-1, 12)


def _key(cost):
    c = np.asarray(cost, np.float64).copy()
    c[np.isnan(c)] = np.inf
    return c


def select_best(cost):
    """index of the lowest final objective (NaN = +inf, ties -> lowest index)."""
    return int(np.argmin(_key(cost)))


def prune_topk(cost, k):
    """indices of the k lowest objectives in ascending (cost, index) order."""
    c = _key(cost)
    order = np.lexsort((np.arange(c.size), c))
    return order[:k].astype(np.int64)

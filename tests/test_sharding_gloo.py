"""world_size-2 (and 3) gloo tests of the multi-GPU host logic (paper_2606_31098_b200/sharding.py) on CPU.
Per-rank compute is stood in for by the oracle on that rank's shard; what is tested is the sharding, the uneven
all-gather and that the gathered result equals the unsharded run."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_31098_b200 import sharding
from tests.small_problems import tiny


def test_shard_bounds_cover_exactly():
    for n in (0, 1, 2, 7, 64, 1210):
        for world in (1, 2, 3, 8):
            cuts = [sharding.shard_bounds(n, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(cuts[r][1] == cuts[r + 1][0] for r in range(world - 1))
            sizes = [e - b for b, e in cuts]
            assert max(sizes) - min(sizes) <= 1 and sorted(sizes, reverse=True) == sizes


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n_hyp, tmp):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import pilot_hypotheses as ph
        from oracle import pilot_oracle as po
        prob = tiny(seed=11, N=60, C=4, n_hyp=n_hyp)
        P = dict(iters=[3], loss="huber", loss_scale=0.3, w_gravity=0.5, min_valid=4)
        mine = sharding.shard_problem(prob, rank, world)
        b, e = mine["shard"]
        assert (b, e) == sharding.shard_bounds(n_hyp, rank, world)
        if e > b:
            o = po.run(po.Bound(mine, P))
            poses, cost = o["poses"], o["cost"]
        else:
            poses, cost = np.zeros((0, 12), np.float32), np.zeros(0, np.float32)
        gp, gc = sharding.gather_results(torch.from_numpy(poses), torch.from_numpy(cost), n_hyp)
        full = po.run(po.Bound(prob, P))
        assert gp.shape == (n_hyp, 12) and gc.shape == (n_hyp,)
        assert np.array_equal(gp.numpy(), full["poses"]) and np.array_equal(gc.numpy(), full["cost"])
        best = ph.select_best(gc.numpy())
        assert best == ph.select_best(full["cost"])
        # every rank ends with the same answer
        t = torch.tensor([float(best)])
        lst = [torch.zeros(1) for _ in range(world)]
        dist.all_gather(lst, t)
        assert all(float(x) == float(best) for x in lst)
        open(os.path.join(tmp, f"ok{rank}"), "w").write("1")
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,n_hyp", [(2, 6), (2, 5), (3, 4), (2, 1)])
def test_sharded_run_equals_unsharded(world, n_hyp, tmp_path):
    mp.spawn(_worker, args=(world, _free_port(), n_hyp, str(tmp_path)), nprocs=world, join=True)
    assert all((tmp_path / f"ok{r}").exists() for r in range(world))


def test_global_best_needs_cuda():
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        sharding.global_best(torch.zeros(2, 12), torch.zeros(2), 2)

"""Multi-GPU: hypotheses are independent for the whole refinement, so the path shards by hypothesis with no
data-path collective. One process per GPU; the scene (pyramid, anchors, DSM) is replicated,
every rank refines a contiguous slice of the hypothesis set, and ONE all-gather of 13 floats per hypothesis
(pose + objective) followed by the arg-min of PAPER.md:168 ends the frame. Host logic only: the refinement and
the arg-min run in the CUDA kernels (binding.select_best); torch.distributed is plumbing (NCCL on GPUs, gloo in
the CPU tests of this module)."""
import numpy as np


def shard_bounds(n, rank, world):
    """Contiguous balanced split of n items: the first n % world ranks get one extra. Returns (begin, end)."""
    assert 0 <= rank < world and n >= 0
    base, extra = divmod(n, world)
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def shard_problem(prob, rank, world):
    """The rank's view of a problem dict: the same scene, its slice of init_poses (and of `units`)."""
    b, e = shard_bounds(int(prob["init_poses"].shape[0]), rank, world)
    q = dict(prob)
    q["init_poses"] = np.ascontiguousarray(prob["init_poses"][b:e])
    H = int(prob["init_poses"].shape[0])
    if "units" in prob and H:
        q["units"] = int(prob["units"]) // H * (e - b)
    q["shard"] = (b, e)
    return q


def gather_results(local_poses, local_cost, n_total, group=None):
    """All-gather of the per-rank results into global hypothesis order.

    local_poses [h_r, 12], local_cost [h_r] (torch tensors on the backend's device: cuda for nccl, cpu for gloo),
    where h_r = the size of shard_bounds(n_total, rank, world). Shards may be uneven: every rank pads to the largest
    shard (cost +inf) so that one fixed-size all_gather serves. Returns (poses [n_total, 12], cost [n_total]) on
    every rank."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    b, e = shard_bounds(n_total, rank, world)
    assert local_poses.shape[0] == e - b == local_cost.shape[0], (local_poses.shape, b, e)
    if not dist.is_initialized():
        return local_poses, local_cost
    h_max = shard_bounds(n_total, 0, world)[1]
    buf = torch.zeros(h_max, 13, dtype=torch.float32, device=local_cost.device)
    buf[:, 12] = float("inf")
    buf[:e - b, :12] = local_poses.reshape(-1, 12)
    buf[:e - b, 12] = local_cost
    out = torch.empty(world * h_max, 13, dtype=torch.float32, device=local_cost.device)
    dist.all_gather_into_tensor(out, buf, group=group)
    keep = [out[r * h_max:r * h_max + (shard_bounds(n_total, r, world)[1] - shard_bounds(n_total, r, world)[0])]
            for r in range(world)]
    allr = torch.cat(keep, 0)
    return allr[:, :12].contiguous(), allr[:, 12].contiguous()


def global_best(local_poses, local_cost, n_total, group=None, stream=None):
    """Gather + the CUDA arg-min kernel: (index into the global set, pose [12], cost [1]) device tensors, identical
    on every rank. CUDA tensors only — there is no CPU path for the selection."""
    from . import binding
    poses, cost = gather_results(local_poses, local_cost, n_total, group)
    return binding.select_best(cost, poses, stream)

#!/usr/bin/env python
"""bench.py — point-hypothesis LM iterations per second of the pilot_refine hot path on B200 (BASELINE.json metric).

A step is one pass of the whole hot path (all levels, all LM iterations, priors, solves)
over one batch of synthetic input. Default workload: config 4 (the configuration north_star's target is quoted
on; 265 MB map > L2). Other workloads (`--config`): config1, config2, config3 (one step = one frame of the
streaming sequence), paper (the paper's own 1210 -> 128 schedule, N=500, K=2/3/4). `--impl reference` times the
CPU oracle on the host cores instead.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "point-hypothesis LM iterations/sec"
UNIT = "point-hyp-iters/s"
LIGHT = ("poses", "cost", "n_valid", "status", "iter_hessian", "iter_gradient", "iter_cost", "iter_lambda")

# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel from the committed `ncu --set full`
# captures of this command (profiles/<file>): the first EVAL pass of a timed step (hypotheses spread over their initial
# poses: the union of their footprints covers the map) and a late pass (hypotheses converged onto one pose). None where
# no capture of that workload exists. Labelled with their source; everything else in the line is measured in this run.
NCU_TRAFFIC = {"config4": {"first_pass_bytes": 420.1e6, "converged_pass_bytes": 31.6e6,
                           "source": "profiles/r2_photo_config4.md"}}


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML during the timed region. NVML is initialised in the constructor
    (before the region) and the thread samples every 5 ms from its first instruction on, so that even a timed region of a
    few milliseconds holds samples taken under load."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.max_mhz = index, False, [], set(), None
        self.nv = self.h = None
        try:
            import pynvml as nv
            nv.nvmlInit()
            self.nv, self.h = nv, nv.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM)
            self.names = {getattr(nv, n): n for n in dir(nv) if n.startswith("nvmlClocksThrottleReason") and
                          isinstance(getattr(nv, n), int)}
        except Exception as e:  # pragma: no cover
            self.reasons.add(f"nvml_error:{type(e).__name__}")

    def sample(self):
        nv, h = self.nv, self.h
        self.sm.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
        r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
        for bit, n in self.names.items():
            if bit and (r & bit) == bit and "All" not in n and "None" not in n:
                self.reasons.add(n.replace("nvmlClocksThrottleReason", ""))

    def run(self):
        if self.nv is None:
            return
        try:
            while not self.stop_flag:
                self.sample()
                time.sleep(0.005)
        except Exception as e:  # pragma: no cover
            self.reasons.add(f"nvml_error:{type(e).__name__}")

    def summary(self):
        sm = sorted(self.sm)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(r for r in self.reasons if r not in ("GpuIdle", "ApplicationsClocksSetting"))}


# ------------------------------------------------------------------ problems

SHUFFLE = {"on": False}


def make_problem(name, rank):
    from paper_2606_31098_b200 import workloads as wl
    prob = wl.make(name)
    if SHUFFLE["on"]:          # a caller that does not sort its anchors: same problem, random anchor order
        rng = np.random.Generator(np.random.PCG64(wl.BASE_SEED + 77))
        for l in range(prob["n_levels"]):
            perm = rng.permutation(prob["points"][l].shape[0])
            prob["points"][l] = np.ascontiguousarray(prob["points"][l][perm])
            prob["ref_feat"][l] = np.ascontiguousarray(prob["ref_feat"][l][perm])
    if rank:  # weak scaling: every rank refines its own shard of hypotheses around the same scene
        rng = np.random.Generator(np.random.PCG64(wl.BASE_SEED + 1000 * rank))
        T = prob["gt_pose"].reshape(3, 4)
        rot, tr = (10.0, 20.0) if name == "config2" else (5.0, 10.0)
        prob["init_poses"] = wl.perturbed_poses(rng, T, prob["init_poses"].shape[0], rot, tr, first_is_gt=False)
    return prob


def gather_bytes_per_launch(prob, H_per_level):
    """4*C*s gather bytes per (anchor, hypothesis) unit x H*N units, averaged over the pass launches of a step."""
    es = 4 if prob["dtype"] == "f32" else 2
    it = prob["params"]["iters"]
    per = [H_per_level[l] * prob["points"][l].shape[0] * 4 * prob["channels"][l] * es
           for l in range(prob["n_levels"]) for _ in range(it[l] + 1)]
    return float(np.mean(per)), len(per)


class Resident:
    """configs 1, 2, 4: one pilot_refine_run per step on inputs resident in HBM (+ the 13-float all-gather and the
    arg-min when sharded over ranks)."""

    def __init__(self, args, rank, local_rank, world):
        import torch
        from paper_2606_31098_b200 import binding
        self.torch, self.binding, self.world, self.dev = torch, binding, world, local_rank
        self.prob = prob = make_problem(args.config, rank)
        self.params = prob["params"]
        self.di = binding.DeviceInputs(prob, local_rank)
        if getattr(args, "sort_anchors", False):
            self.di.sort_anchors()                       # pilot_refine_sort_anchors: Morton order on the device
        self.ref = binding.Refiner.for_inputs(self.di, self.params, local_rank)
        if args.chunk:
            self.ref.set_chunk(args.chunk)
        self.ref.set_exec_mode(args.mode, args.cluster)
        self.ref.set_math_mode(args.math)
        self.H = prob["init_poses"].shape[0]
        self.units = prob["units"]
        self.bytes_per_launch, self.pass_launches = gather_bytes_per_launch(prob, [self.H] * prob["n_levels"])
        self.args = args

    def step(self, stream):
        self.out = self.ref.run(self.di, self.params, stream, LIGHT)
        if self.torch.distributed.is_initialized():
            from paper_2606_31098_b200 import sharding
            self.best = sharding.global_best(self.out["poses"], self.out["cost"], self.world * self.H, stream=stream)

    @property
    def launches(self):
        return self.ref.last_launches + (1 if self.torch.distributed.is_initialized() else 0)

    def visible_evals(self, stream):
        """(visible, all) (anchor, hypothesis) unit evaluations of one step: every EVAL pass of every level."""
        it = self.params["iters"]
        total = sum(self.H * self.prob["points"][l].shape[0] * (it[l] + 1) for l in range(self.prob["n_levels"]))
        return self.ref.last_visible_evals(stream), total

    def plan(self):
        return self.ref.last_plan()

    def check(self):
        cost = self.out["cost"].cpu().numpy()
        assert np.isfinite(cost).any(), "no hypothesis ended with a finite cost"

    def config(self):
        p = self.prob
        return {"hypotheses_per_gpu": self.H, "points": [int(q.shape[0]) for q in p["points"]],
                "channels": p["channels"], "feat_dtype": p["dtype"], "iters": self.params["iters"],
                "levels": p["n_levels"]}

    def map_bytes(self):
        return sum(int(np.asarray(q).nbytes) for q in self.prob["query_feat"])

    def e2e(self, stream, n):
        """Host-buffer path: pinned host inputs -> H2D -> run -> D2H of every output, per step, pipelined over steps."""
        binding = self.binding
        hi = binding.DeviceInputs(self.prob, self.dev, host=True)
        href = binding.Refiner.for_inputs(hi, self.params, self.dev, host_path=True)
        if self.args.chunk:
            href.set_chunk(self.args.chunk)
        href.set_exec_mode(self.args.mode, self.args.cluster)
        href.set_math_mode(self.args.math)
        T = sum(self.params["iters"])
        d2h = self.H * (48 + 4 + 4 + 4) + T * self.H * (144 + 24 + 4 + 4)
        href.run(hi, self.params, stream, LIGHT)
        self.torch.cuda.synchronize(self.dev)
        # every step uploads all of its inputs and reads back all of its outputs; step k+1 is submitted before step k
        # is waited for, so its H2D copy overlaps step k's kernels (pilot_refine_submit_host / _wait_host)
        t0 = time.perf_counter()
        href.submit(hi, self.params, stream, LIGHT)
        for i in range(n):
            if i + 1 < n:
                href.submit(hi, self.params, stream, LIGHT)
            res = href.wait()
            assert np.isfinite(res["cost"].numpy()).any()
        dt = time.perf_counter() - t0
        href.close()
        return dt, int(hi.h2d_bytes), int(d2h)

    def cpu_problem(self):
        return self.prob

    def close(self):
        self.ref.close()


class Streaming:
    """config 3: one step = one frame. `value`: seed -> run -> arg-min on frames resident in HBM (a ring of 4);
    `e2e`: pilot_refine_sequence_* streaming every frame from host memory on the side stream."""

    RING = 4

    def __init__(self, args, rank, local_rank, world):
        import torch
        from paper_2606_31098_b200 import binding, workloads as wl
        self.torch, self.binding, self.world, self.dev, self.wl = torch, binding, world, local_rank, wl
        self.seq = seq = wl.Config3Sequence()
        self.params = seq.params
        self.frames = [seq.frame(i + 1) for i in range(self.RING)]
        d = torch.device("cuda", local_rank)
        self.di = [binding.DeviceInputs(f, local_rank) for f in self.frames]
        self.offsets = torch.from_numpy(seq.offsets).to(d)
        self.priors = [torch.from_numpy(seq.gt_pose(i).reshape(-1).astype(np.float32)).to(d) for i in range(self.RING)]
        self.seeds = torch.empty(seq.H, 12, dtype=torch.float32, device=d)
        for di in self.di:
            di.inp.n_hypotheses, di.n_hyp = seq.H, seq.H
            di.inp.init_poses_dev = self.seeds.data_ptr()
        self.ref = binding.Refiner.for_inputs(self.di[0], self.params, local_rank)
        self.ref.set_exec_mode(args.mode, args.cluster)
        self.ref.set_math_mode(args.math)
        self.H, self.units, self.i = seq.H, seq.units_per_frame, 0
        self.prob = dict(self.frames[0], params=self.params)
        self.bytes_per_launch, self.pass_launches = gather_bytes_per_launch(self.prob, [self.H] * 3)

    def step(self, stream):
        k = self.i % self.RING
        self.i += 1
        b = self.binding
        b.seed_hypotheses(self.priors[k], self.offsets, "camera", out=self.seeds, stream=stream)
        self.out = self.ref.run(self.di[k], self.params, stream, ("poses", "cost", "n_valid", "status"))
        self.best = b.select_best(self.out["cost"], self.out["poses"], stream)

    @property
    def launches(self):
        return self.ref.last_launches + 2

    def visible_evals(self, stream):
        total = sum(self.H * self.seq.N * (k + 1) for k in self.seq.iters)
        return self.ref.last_visible_evals(stream), total

    def plan(self):
        return self.ref.last_plan()

    def check(self):
        gt = self.seq.gt_pose((self.i - 1) % self.RING + 1).reshape(-1)
        err = np.linalg.norm(self.best[1].cpu().numpy().reshape(3, 4)[:, 3] - gt.reshape(3, 4)[:, 3])
        assert err < 1.0, f"frame estimate {err:.2f} m from the ground truth"

    def config(self):
        s = self.seq
        return {"hypotheses_per_gpu": s.H, "points": [s.N] * 3, "channels": [32] * 3, "feat_dtype": "bf16",
                "iters": s.iters, "levels": 3, "step": "one frame", "resident_ring": self.RING}

    def map_bytes(self):
        return sum(int(np.asarray(q).nbytes) for q in self.frames[0]["query_feat"])

    def e2e(self, stream, n):
        b, s = self.binding, self.seq
        n = max(n, 30)
        L = s.LEVELS
        S = b.Sequence(3, [l[0] for l in L], [l[1] for l in L], [l[2] for l in L], "bf16", s.H, s.N, sum(s.iters),
                       s.offsets, s.dsm, s.origin, s.gsd, s.gravity_world, n + 1)
        ring = [b.make_frame(f, pin=True) for f in self.frames]          # page-locked once; every frame is still uploaded
        frames = (ring * (n // self.RING + 2))[:n + 1]
        S.set_prior(s.gt_pose(0).reshape(-1), stream)
        S.upload(frames[0]); S.upload(frames[1]); S.step(self.params, stream)      # warm-up frame
        self.torch.cuda.synchronize(self.dev)
        t0 = time.perf_counter()
        for i in range(1, n + 1):
            if i + 1 <= n:
                S.upload(frames[i + 1])
            S.step(self.params, stream)
        rows = S.results(1, n, stream)                                              # D2H of the n result rows + sync
        dt = time.perf_counter() - t0
        assert np.isfinite(rows[:, 12]).all()
        S.close()
        self.e2e_steps = n
        return dt, int(frames[0][2]), 64

    def cpu_problem(self):
        from oracle import pilot_hypotheses as ph
        seeds = ph.seed_hypotheses(self.seq.gt_pose(0).reshape(-1), self.seq.offsets, ph.SEED_CAMERA)
        return self.wl.with_poses(self.prob, seeds)

    def close(self):
        self.ref.close()


class PaperSchedule:
    """The paper's own per-frame problem: 1210 grid hypotheses on the coarse level, top 128
    on the medium and fine levels, N=500, K=2/3/4. Context for the paper's 43.82 ms optimizer time (RTX 5090)."""

    def __init__(self, args, rank, local_rank, world):
        import torch
        from paper_2606_31098_b200 import binding, workloads as wl
        self.torch, self.binding, self.world, self.dev = torch, binding, world, local_rank
        self.prob = prob = wl.paper_frame()
        self.params = prob["params"]
        self.off = binding.grid_offsets(prob["grid"][0], prob["grid"][1], prob["grid"][2], -prob["gravity_world"])
        self.di = binding.DeviceInputs(prob, local_rank)
        self.pr = binding.PrunedRefiner(self.di, self.params, self.off, prob["keep"], "world", local_rank)
        self.pr.ref.set_exec_mode(args.mode, args.cluster)
        self.pr.ref.set_math_mode(args.math)
        self.prior = torch.from_numpy(prob["prior_pose"]).to(torch.device("cuda", local_rank))
        self.H0, self.keep, self.units = self.off.shape[0], prob["keep"], prob["units"]
        self.bytes_per_launch, self.pass_launches = gather_bytes_per_launch(prob, [self.H0, self.keep, self.keep])

    def step(self, stream):
        self.out = self.pr.run(self.prior, stream)

    @property
    def launches(self):
        return self.pr.launches

    def visible_evals(self, stream):
        it = self.params["iters"]
        self.pr.run(self.prior, stream, count_visible=True)
        total = self.H0 * 500 * (it[0] + 1) + self.keep * 500 * ((it[1] + 1) + (it[2] + 1))
        return sum(self.pr.visible_evals), total

    def plan(self):
        return self.pr.ref.last_plan()

    def check(self):
        gt = self.prob["gt_pose"].reshape(3, 4)[:, 3]
        err = np.linalg.norm(self.out["best_pose"].cpu().numpy().reshape(3, 4)[:, 3] - gt)
        assert err < 0.5, f"estimate {err:.2f} m from the ground truth"

    def config(self):
        p = self.prob
        return {"hypotheses_per_gpu": [self.H0, self.keep, self.keep], "points": [500] * 3, "channels": p["channels"],
                "feat_dtype": p["dtype"], "iters": self.params["iters"], "levels": 3,
                "schedule": "1210 (x,y,yaw) grid -> coarse level -> top 128 -> medium, fine -> arg-min",
                "paper_context": "paper: optimizer 43.82 ms per frame on an RTX 5090 (PAPER.md:473), another machine"}

    def map_bytes(self):
        return sum(int(np.asarray(q).nbytes) for q in self.prob["query_feat"])

    def e2e(self, stream, n):
        """Per step one C call through HOST buffers (pilot_refine_submit_pruned_host): H2D of every input of the frame, the
        whole 1210 -> 128 schedule, D2H of the selected pose, objective and grid index; frame k+1 is submitted before
        frame k is waited for, so its upload overlaps frame k's kernels."""
        torch, b = self.torch, self.binding
        hi = b.DeviceInputs(self.prob, self.dev, host=True)
        ph = b.PrunedHostRefiner(hi, self.params, self.off, self.keep, "world", self.dev)
        n = max(n, 20)
        gt = self.prob["gt_pose"].reshape(3, 4)[:, 3]
        ph.submit(self.prob["prior_pose"], stream); ph.wait()                     # warm-up frame
        torch.cuda.synchronize(self.dev)
        t0 = time.perf_counter()
        ph.submit(self.prob["prior_pose"], stream)
        for i in range(n):
            if i + 1 < n:
                ph.submit(self.prob["prior_pose"], stream)
            r = ph.wait()
            assert np.linalg.norm(r["pose"].numpy().reshape(3, 4)[:, 3] - gt) < 0.5
        dt = time.perf_counter() - t0
        ph.close()
        self.e2e_steps = n
        return dt, int(hi.h2d_bytes) + 48, 56

    def cpu_problem(self):
        return None

    def cpu_time(self, cores):
        from oracle import pilot_hypotheses as ph
        from oracle import pilot_oracle as po
        from paper_2606_31098_b200 import workloads as parity       # levels_slice: dict slicing only
        p = self.prob
        t0 = time.perf_counter()
        seeds = ph.seed_hypotheses(p["prior_pose"], self.off, ph.SEED_WORLD)
        c0 = po.run(po.Bound(parity.levels_slice(p, 0, 1, seeds)), n_threads=cores)
        keep = ph.prune_topk(c0["cost64"], p["keep"])
        c1 = po.run(po.Bound(parity.levels_slice(p, 1, 3, c0["poses64"][keep])), n_threads=cores)
        ph.select_best(c1["cost64"])
        dt = time.perf_counter() - t0
        return p["units"] / dt, f"the whole 1210 -> 128 schedule of one frame, {dt:.1f} s", min(cores, c0["threads"])

    def close(self):
        self.pr.close()


WORKLOADS = {"config1": Resident, "config2": Resident, "config4": Resident, "config3": Streaming,
             "paper": PaperSchedule}


# ------------------------------------------------------------------ CPU oracle legs

def oracle_sample(prob, cores, budget_hyps=None):
    """Time the oracle as it stands on a strided subset of hypotheses (full N and K). Returns (units/s, desc, threads)."""
    from oracle import pilot_oracle as po
    H = prob["init_poses"].shape[0]
    n = min(H, budget_hyps or 4 * cores)
    stride = max(1, H // n)
    idx = list(range(0, H, stride))
    b = po.Bound(prob)
    t0 = time.perf_counter()
    o = po.run(b, hyp_begin=0, hyp_step=stride, n_threads=cores)
    dt = time.perf_counter() - t0
    units = prob["units"] // H * len(idx)
    threads = min(o["threads"], len(idx))
    return units / dt, f"{len(idx)} of {H} hypotheses (stride {stride}), full N and K, {dt:.1f} s", threads


def reference_problem(name):
    from paper_2606_31098_b200 import workloads as wl
    if name == "config3":
        from oracle import pilot_hypotheses as ph
        seq = wl.Config3Sequence()
        f = seq.frame(1)
        return wl.with_poses(f, ph.seed_hypotheses(seq.gt_pose(0).reshape(-1), seq.offsets, ph.SEED_CAMERA))
    if name == "paper":
        from oracle import pilot_hypotheses as ph
        parity = wl                                                  # levels_slice: dict slicing only
        p = wl.paper_frame()
        off = ph.grid_offsets(p["grid"][0], p["grid"][1], p["grid"][2], -p["gravity_world"])
        q = parity.levels_slice(p, 0, 1, ph.seed_hypotheses(p["prior_pose"], off, ph.SEED_WORLD))
        q["units"] = int(off.shape[0] * 500 * p["params"]["iters"][0])
        return q
    return make_problem(name, 0)


def run_reference(args, rank):
    if rank != 0:
        return
    prob = reference_problem(args.config)
    cores = os.cpu_count() or 1
    vals, times, desc, threads = [], [], "", 1
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        v, desc, threads = oracle_sample(prob, cores, budget_hyps=max(2, min(cores, 16)))
        if i >= args.warmup:
            vals.append(v)
            times.append(time.perf_counter() - t0)
    value = float(np.mean(vals))
    H = prob["init_poses"].shape[0]
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * float(np.mean(times)), "ms_per_step_extrapolated_to_full_workload": 1e3 * prob["units"] / value,
            "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.config, "hypotheses": H, "points": int(prob["points"][0].shape[0]),
                       "note": "CPU oracle (oracle/pilot_oracle.c); a step = a bounded hypothesis sample of the workload "
                               "(see cpu_baseline.sample): ms_per_step is the measured time of that sample, value the "
                               "rate, which does not depend on the sample because hypotheses are independent"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------ measurement

def measure(W, steps, warmup, stream, local_rank, world, use_dist, flush):
    """W untimed warm-up steps, then `steps` timed steps (CUDA events on the launching stream, a barrier and a device
    synchronise on both sides, max over ranks), the SM clock sampled during the timed region."""
    import torch
    import torch.distributed as dist

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize(local_rank)

    for _ in range(warmup):
        W.step(stream)
    barrier()
    launches = W.launches
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    barrier()
    for s, e in ev:
        if flush is not None:
            flush.fill_(1)                 # evict the maps from L2 between timed steps (outside the events)
        s.record(stream)
        W.step(stream)
        e.record(stream)
    barrier()
    sampler.stop_flag = True
    sampler.join()
    total_ms = sum(s.elapsed_time(e) for s, e in ev)
    t = torch.tensor([total_ms], dtype=torch.float64, device=f"cuda:{local_rank}")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms = float(t.item())
    W.check()
    vis, tot = W.visible_evals(stream)
    return {"ms_per_step": total_ms / steps, "value": world * W.units * steps / (total_ms * 1e-3), "launches": launches,
            "clocks": sampler.summary(), "visible_evals": vis, "all_evals": tot}


def measure_graph(W, steps, local_rank, flush):
    """The same step captured once into a CUDA graph and replayed (what a serving loop does with a launch-bound step: the
    library's calls are capturable - no allocation, no host synchronisation). Returns ms per step, or None if the capture
    fails. Timed like measure(): CUDA events around every replay, the L2 flush outside them."""
    import torch
    try:
        side = torch.cuda.Stream(device=local_rank)
        side.wait_stream(torch.cuda.current_stream(local_rank))
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            W.step(side)                                   # allocations of the binding settle before the capture
            side.synchronize()
            with torch.cuda.graph(g, stream=side):
                W.step(side)
        torch.cuda.synchronize(local_rank)
        for _ in range(3):
            g.replay()
        torch.cuda.synchronize(local_rank)
        cur = torch.cuda.current_stream(local_rank)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for s, e in ev:
            if flush is not None:
                flush.fill_(1)
            s.record(cur)
            g.replay()
            e.record(cur)
        torch.cuda.synchronize(local_rank)
        W.check()
        return sum(s.elapsed_time(e) for s, e in ev) / steps
    except Exception as ex:                                # noqa: BLE001  (reported, not fatal: the stream-launched figure stands)
        sys.stderr.write(f"[bench] CUDA-graph leg skipped: {ex}\n")
        return None


def roofline_of(W, m, name, peaks, hbm_peak, hbm_src, map_bytes, l2_bytes):
    """The dominant kernel's roofline. What binds is the gather of the taps from L2 into the SMs (the
    maps are L2-resident, or - config 4 - the union of the co-resident CTAs' footprints is: 30-420 MB of DRAM traffic per
    pass against GBs of taps), so `bound` is "l2-gather": achieved = tap bytes of the VISIBLE units (4*C*s each, SURVEY's
    per-unit figure; invisible units move nothing) per EVAL pass / the pass's share of the step time, peak = the same
    access shape without arithmetic from an L2-resident buffer, measured in this run by pilot_refine_probe_unit_gather.
    north_star's "HBM-gather roofline" (every tap byte of every unit from HBM, no reuse) is reported beside it."""
    es = 4 if W.prob["dtype"] == "f32" else 2
    C_last = W.prob["channels"][-1]
    unit_bytes = 4 * C_last * es
    passes = W.pass_launches
    pass_s = m["ms_per_step"] * 1e-3 / passes          # seed / init / select kernels and launch gaps included: conservative
    vis_per_pass, all_per_pass = m["visible_evals"] / passes, m["all_evals"] / passes
    achieved = vis_per_pass * unit_bytes / pass_s / 1e9
    achieved_all = all_per_pass * unit_bytes / pass_s / 1e9
    pk = peaks.get(C_last * es) if peaks else None
    mma, res = W.plan()
    r = {"bound": "l2-gather", "achieved": achieved, "peak": pk["l2_ldg_gbs"] if pk else None, "unit": "GB/s",
         "frac": achieved / pk["l2_ldg_gbs"] if pk and pk["l2_ldg_gbs"] else None,
         "traffic": None, "kernel": "lm_resident_kernel (K+1 passes per launch)" if res else "photo_pass_kernel (one pass per launch)",
         "algorithmic_bytes_per_pass": vis_per_pass * unit_bytes, "pass_ms": pass_s * 1e3, "eval_passes_per_step": passes,
         "bytes_per_visible_unit": unit_bytes, "visible_fraction": m["visible_evals"] / max(1, m["all_evals"]),
         "contraction": "mma.sync (tensor cores)" if mma else "FFMA2", "levels_on_tensor_cores": mma, "levels_resident": res,
         "peak_source": "pilot_refine_probe_unit_gather: unit-shaped random gather (2x2 pixels + reference row, four lanes per "
                        "unit) from a 16 MiB buffer, measured in this run" if pk else "probe skipped",
         "hbm_no_reuse": {"achieved_all_units": achieved_all, "achieved_visible_units": achieved, "peak": hbm_peak, "unit": "GB/s",
                          "frac_all_units": achieved_all / hbm_peak, "frac_visible_units": achieved / hbm_peak,
                          "peak_source": hbm_src,
                          "note": "north_star's HBM-gather roofline: 4*C*s bytes per unit as if every tap crossed HBM once "
                                  "(all H*N units, SURVEY.md §8(d).1; target >= 0.60 on config 4). HBM does not bind: the "
                                  "taps are served from L2 (see traffic), so this ratio may exceed 1"}}
    t = NCU_TRAFFIC.get(name)
    if t:
        r["traffic"] = t["first_pass_bytes"]
        r["traffic_converged_pass"] = t["converged_pass_bytes"]
        r["traffic_source"] = t["source"] + " (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum of one launch)"
    if pk:
        r["gather_peaks"] = pk
    compulsory = float(map_bytes) / max(1, W.prob["n_levels"])          # one level's map read once per pass
    model = {"t_hbm_compulsory_ms": compulsory / (hbm_peak * 1e9) * 1e3,
             "t_hbm_first_pass_ms": t["first_pass_bytes"] / (hbm_peak * 1e9) * 1e3 if t else None,
             "t_l2_gather_ms": vis_per_pass * unit_bytes / (pk["l2_ldg_gbs"] * 1e9) * 1e3 if pk and pk["l2_ldg_gbs"] else None,
             "t_pass_ms": pass_s * 1e3}
    terms = {k: v for k, v in model.items() if k != "t_pass_ms" and v}
    if terms:
        model["binds"] = max(terms, key=terms.get)
        model["t_model_over_t_pass"] = max(terms.values()) / model["t_pass_ms"]
    r["model"] = model
    return r


def gather_peaks(binding, px_sizes, local_rank):
    """The build's own micro-benchmark for every pixel size the workloads use."""
    out = {}
    for px in sorted(set(px_sizes)):
        if px not in (64, 128):
            continue
        out[px] = {"px_bytes": px,
                   "l2_ldg_gbs": binding.probe_unit_gather(16 << 20, px, 0, 5, local_rank),
                   "l2_staged_bulk_gbs": binding.probe_unit_gather(16 << 20, px, 1, 5, local_rank),
                   "hbm_ldg_gbs": binding.probe_unit_gather(4 << 30, px, 0, 3, local_rank),
                   "note": "GB/s of tap bytes (4 pixels per unit; the reference row moves too, uncounted). ldg = the kernel's "
                           "access shape; staged_bulk = cp.async.bulk into shared memory + LDS.128 (north_star's staged "
                           "variant, measured and not adopted: profiles/r2_staged_vs_ldg.md)"}
    return out


def dtype_string(W):
    mma, _ = W.plan()
    d = W.prob["dtype"]
    if d == "f32":
        return "f32"
    if mma:
        return d + (" storage; first differences in %s, products on mma.sync with f32 accumulate" % d) + \
            "; f32 projection (visibility decided in f64) and lift, f64 6x6 solve"
    return d + " storage, f32 FFMA2 contraction; f32 lift, f64 projection and 6x6 solve"


def run_workload(name, args, rank, local_rank, world, use_dist, stream, steps, peaks, hbm, l2_bytes, with_e2e, with_cpu):
    import torch
    import torch.distributed as dist
    if name != args.config:                # one of the default run's other workloads: heuristics only
        args = argparse.Namespace(**vars(args))
        args.config, args.mode, args.math, args.chunk, args.cluster = name, "auto", "auto", 0, 0
    W = WORKLOADS[name](args, rank, local_rank, world)
    map_bytes = W.map_bytes()
    need_flush = map_bytes <= l2_bytes
    flush = torch.empty(max(2 * l2_bytes, 1 << 28), dtype=torch.uint8, device=f"cuda:{local_rank}") if need_flush else None
    warmup = max(3, args.warmup)
    m = measure(W, steps, warmup, stream, local_rank, world, use_dist, flush)
    roof = roofline_of(W, m, name, peaks, hbm[0], hbm[1], map_bytes, l2_bytes)
    e2e = None
    if with_e2e:
        n_e2e = max(1, min(steps, 10))
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize(local_rank)
        dt, h2d, d2h = W.e2e(stream, n_e2e)
        n_e2e = getattr(W, "e2e_steps", n_e2e)
        tt = torch.tensor([dt], dtype=torch.float64, device=f"cuda:{local_rank}")
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e = {"value": world * W.units * n_e2e / float(tt.item()), "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": n_e2e}
    cpu = None
    if with_cpu and rank == 0 and world == 1:
        cores = os.cpu_count() or 1
        cp = W.cpu_problem()
        v, desc, threads = oracle_sample(cp, cores) if cp is not None else W.cpu_time(cores)
        cpu = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc}
        if cp is not None:                 # the single-thread figure BASELINE.md §3 plans, on a smaller sample
            v1, d1, _ = oracle_sample(cp, 1, budget_hyps=2)
            cpu["value_1_core"] = v1
            cpu["sample_1_core"] = d1
    cfg = {"workload": name, "exec_mode": args.mode, "math_mode": args.math}
    cfg.update(W.config())
    cfg.update({"map_bytes": map_bytes, "l2_bytes": int(l2_bytes),
                "l2_policy": "L2 flushed between timed steps" if need_flush else "inputs larger than L2"})
    res = {"ms_per_step": m["ms_per_step"], "value": m["value"], "steps": steps, "warmup": warmup, "dtype": dtype_string(W),
           "config": cfg, "roofline": roof, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(m["launches"] * steps),
           "clocks": m["clocks"]}
    # last, after everything the line needs has been measured: the same step replayed from a CUDA graph
    graph_ms = measure_graph(W, steps, local_rank, flush) if (name != "config3" and world == 1) else None
    if graph_ms is not None:
        res["cuda_graph"] = {"ms_per_step": graph_ms, "value": W.units / (graph_ms * 1e-3), "unit": UNIT,
                             "note": "the same step captured once and replayed (launch gaps removed); ms_per_step above is stream-launched"}
    W.close()
    del W, flush
    torch.cuda.empty_cache()
    return res


# ------------------------------------------------------------------ main

def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="config4", choices=sorted(WORKLOADS))
    ap.add_argument("--chunk", type=int, default=0, help="anchors per CTA of the pass kernel (0 = heuristic)")
    ap.add_argument("--mode", default="auto", choices=["auto", "passes", "resident", "split"], help="launch strategy (pilot_exec_mode)")
    ap.add_argument("--math", default="auto", choices=["auto", "fp32", "mma"], help="per-unit contraction (pilot_math_mode)")
    ap.add_argument("--cluster", type=int, default=0, help="CTAs per hypothesis of the resident kernel (0 = heuristic)")
    ap.add_argument("--shuffle-anchors", action="store_true", help="hand the anchors over in a random order instead of the "
                    "generator's Morton order (config1/2/4): measures what the caller's ordering is worth")
    ap.add_argument("--sort-anchors", action="store_true", help="put the anchors in Morton order with pilot_refine_sort_anchors "
                    "before the timed region (with --shuffle-anchors: what the library's own ordering recovers)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-probe", action="store_true", help="skip the gather-peak micro-benchmark")
    ap.add_argument("--no-others", action="store_true", help="default run only: skip the other workloads' lines")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        return run_reference(args, rank)
    SHUFFLE["on"] = args.shuffle_anchors

    import torch
    import torch.distributed as dist
    from paper_2606_31098_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    use_dist = world > 1 or "RANK" in os.environ        # under torchrun (also with one rank) the NCCL path runs
    if use_dist:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    stream = torch.cuda.current_stream(local_rank)
    l2_bytes = torch.cuda.get_device_properties(local_rank).L2_cache_size
    hbm = load_peaks()
    default_run = args.config == "config4" and world == 1 and not args.no_others and not args.shuffle_anchors and not args.sort_anchors
    peaks = None
    if rank == 0 and not args.no_probe:
        peaks = gather_peaks(binding, [64, 128] if default_run else [128 if args.config in ("config2", "config4") else 64], local_rank)
    main_res = run_workload(args.config, args, rank, local_rank, world, use_dist, stream, args.steps, peaks, hbm, l2_bytes,
                            not args.no_e2e, not args.no_cpu_baseline)
    others = None
    if default_run and rank == 0:
        # the other BASELINE.json configs and the paper's own schedule, in the same process and under the same clock
        # sampling, so that the driver's record carries all five (each is well under a second of GPU time per step)
        others = {}
        for name in ("config1", "config2", "config3", "paper"):
            try:
                r = run_workload(name, args, rank, local_rank, world, use_dist, stream, min(args.steps, 10), peaks, hbm, l2_bytes,
                                 not args.no_e2e, False)
            except Exception as ex:            # noqa: BLE001  (the headline line must still be printed)
                others[name] = {"error": f"{type(ex).__name__}: {ex}"}
                continue
            others[name] = {k: r[k] for k in ("ms_per_step", "value", "steps", "dtype", "e2e", "gpu_launches", "clocks")}
            others[name]["config"] = {k: r["config"][k] for k in ("hypotheses_per_gpu", "points", "channels", "iters", "l2_policy")}
            others[name]["roofline"] = {k: r["roofline"].get(k) for k in ("bound", "achieved", "peak", "unit", "frac", "kernel",
                                                                          "visible_fraction", "contraction", "pass_ms")}
            others[name]["roofline"]["hbm_no_reuse_frac_all_units"] = r["roofline"]["hbm_no_reuse"]["frac_all_units"]
            if "cuda_graph" in r:
                others[name]["cuda_graph"] = r["cuda_graph"]

    if rank == 0:
        cfg = main_res["config"]
        cfg["sharding"] = ("hypotheses across ranks, no data-path collective; one 13-float-per-hypothesis "
                           "all-gather + arg-min ends the step when n_gpus > 1")
        if args.shuffle_anchors or args.sort_anchors:
            cfg["anchor_order"] = ("random permutation (--shuffle-anchors)" if args.shuffle_anchors else "generator's order") + \
                (", then pilot_refine_sort_anchors (Morton order on the device)" if args.sort_anchors else "")
        line = {"metric": METRIC, "value": main_res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": main_res["warmup"], "ms_per_step": main_res["ms_per_step"], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": main_res["dtype"], "data": "synthetic", "config": cfg,
                "roofline": main_res["roofline"], "cpu_baseline": main_res["cpu_baseline"], "e2e": main_res["e2e"],
                "gpu_launches": main_res["gpu_launches"], "clocks": main_res["clocks"]}
        if "cuda_graph" in main_res:
            line["cuda_graph"] = main_res["cuda_graph"]
        if others is not None:
            line["other_workloads"] = others
        print(json.dumps(line))
    if use_dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

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

# dram__bytes_read.sum + dram__bytes_write.sum per photo_pass_kernel launch from the committed `ncu --set full`
# capture of this command (profiles/r1h_photo_config4.md, r1g before the 1536-anchor chunks; r1d for --math fp32: the same 34-37 MB); None where no
# capture of that workload exists.
NCU_TRAFFIC_BYTES = {"config4": 35.5e6, "config2": 18.0e6}    # config 2: profiles/r1g_photo_config2.md
# From the same captures, per (anchor, hypothesis) unit-evaluation of the pass kernel at C = 64 bf16: warp instructions
# and L1 data-pipe wavefronts (l1tex__data_pipe_lsu_wavefronts: global + shared + local + shuffles). C = 32: the
# cluster-resident kernel (profiles/r1c_resident_small_workloads.md).
NCU_PER_UNIT = {("mma", 64): {"inst": 30.5, "l1_wavefronts": 10.4, "source": "profiles/r1g_photo_config4.md"},
                ("fp32", 64): {"inst": 47.5, "l1_wavefronts": 11.4, "source": "profiles/r1d_photo_config4.md"},
                ("fp32", 32): {"inst": 32.7, "l1_wavefronts": None, "source": "profiles/r1c_resident_small_workloads.md"}}


def contraction_used(args, prob, H):
    """Which per-unit contraction the library takes for this run (pilot_math_mode, include/pilot_refine.h): mirrors
    AUTO's rule so that the roofline constants match the kernel that ran."""
    C, N = prob["channels"][-1], max(p.shape[0] for p in prob["points"])
    applies = prob["dtype"] != "f32" and C in (16, 32, 64, 128)
    if args.math == "fp32" or not applies:
        return "fp32"
    if args.math == "mma":
        return "mma"
    resident = args.mode == "resident" or (args.mode == "auto" and H * N <= 1500000 and H <= 296)
    return "mma" if C >= 64 and not resident else "fp32"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML during the timed region."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.max_mhz = index, False, [], set(), None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {getattr(nv, n): n for n in dir(nv) if n.startswith("nvmlClocksThrottleReason") and
                     isinstance(getattr(nv, n), int)}
            while not self.stop_flag:
                self.sm.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, n in names.items():
                    if bit and (r & bit) == bit and "All" not in n and "None" not in n:
                        self.reasons.add(n.replace("nvmlClocksThrottleReason", ""))
                time.sleep(0.05)
        except Exception as e:  # pragma: no cover
            self.reasons.add(f"nvml_error:{type(e).__name__}")

    def summary(self):
        sm = sorted(self.sm)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(r for r in self.reasons if r not in ("GpuIdle", "ApplicationsClocksSetting"))}


# ------------------------------------------------------------------ problems

def make_problem(name, rank):
    from paper_2606_31098_b200 import workloads as wl
    prob = wl.make(name)
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
        """Per step: pinned host inputs -> device (torch copies on the same stream), the five-call schedule, the
        selected pose and objective back to the host."""
        torch, b = self.torch, self.binding
        hi = b.DeviceInputs(self.prob, self.dev, host=True)
        prior_h = torch.from_numpy(self.prob["prior_pose"]).pin_memory()

        def once():
            with torch.cuda.stream(stream):
                for src, dst in zip(hi.keep, self.di.keep):
                    dst.copy_(src, non_blocking=True)
                self.prior.copy_(prior_h, non_blocking=True)
            o = self.pr.run(self.prior, stream)
            with torch.cuda.stream(stream):
                return o["best_pose"].cpu(), o["best_cost"].cpu()
        once()
        torch.cuda.synchronize(self.dev)
        t0 = time.perf_counter()
        for _ in range(n):
            once()
        torch.cuda.synchronize(self.dev)
        return time.perf_counter() - t0, int(hi.h2d_bytes) + 48, 52

    def cpu_problem(self):
        return None

    def cpu_time(self, cores):
        from oracle import pilot_hypotheses as ph
        from oracle import pilot_oracle as po
        from tests import parity
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
        from tests import parity
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
    vals, desc, threads = [], "", 1
    for i in range(args.warmup + args.steps):
        v, desc, threads = oracle_sample(prob, cores, budget_hyps=max(2, min(cores, 16)))
        if i >= args.warmup:
            vals.append(v)
    value = float(np.mean(vals))
    H = prob["init_poses"].shape[0]
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * prob["units"] / value, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.config, "hypotheses": H, "points": int(prob["points"][0].shape[0]),
                       "note": "CPU oracle (oracle/pilot_oracle.c) on a bounded hypothesis sample per step; "
                               "ms_per_step extrapolated to the whole workload"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


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
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-probe", action="store_true", help="skip the gather-peak micro-benchmark")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        return run_reference(args, rank)

    import torch
    import torch.distributed as dist
    from paper_2606_31098_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    use_dist = world > 1 or "RANK" in os.environ        # under torchrun (also with one rank) the NCCL path runs
    if use_dist:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    W = WORKLOADS[args.config](args, rank, local_rank, world)
    stream = torch.cuda.current_stream(local_rank)
    map_bytes = W.map_bytes()
    l2_bytes = torch.cuda.get_device_properties(local_rank).L2_cache_size
    need_flush = map_bytes <= l2_bytes
    flush = torch.empty(max(2 * l2_bytes, 1 << 28), dtype=torch.uint8, device=f"cuda:{local_rank}") if need_flush else None
    warmup = max(3, args.warmup)

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize(local_rank)

    for _ in range(warmup):
        W.step(stream)
    barrier()
    launches_per_step = W.launches
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
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
    units = W.units
    value = world * units * args.steps / (total_ms * 1e-3)
    W.check()

    # ---- roofline of the dominant kernel (photo_pass_kernel): algorithmic gather bytes per launch / launch time
    launch_s = (total_ms * 1e-3 / args.steps) / W.pass_launches   # init / seed / select kernels and gaps included: conservative
    peak, peak_src = load_peaks()
    achieved = W.bytes_per_launch / launch_s / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": NCU_TRAFFIC_BYTES.get(args.config), "kernel": "photo_pass_kernel",
                "algorithmic_bytes_per_launch": W.bytes_per_launch, "launch_ms": launch_s * 1e3,
                "peak_source": peak_src,
                "note": "4*C*s gather bytes per (anchor,hypothesis) unit x H*N units per launch (north_star's "
                        "HBM-gather roofline, no-reuse model); the taps are served through L2, so achieved may "
                        "exceed the HBM copy peak when L2 reuse is high"}
    # the bound that actually applies: plain fp32 arithmetic. Algorithmic flops per unit-evaluation =
    # 2*(19*C + 120); peak = SMs x 128 fp32 lanes x 2 flop x max SM clock
    prop = torch.cuda.get_device_properties(local_rank)
    flops_per_launch = W.bytes_per_launch / (4 * W.prob["channels"][-1] * (4 if W.prob["dtype"] == "f32" else 2)) \
        * 2 * (19 * W.prob["channels"][-1] + 120)
    alu_peak = prop.multi_processor_count * 128 * 2 * 1.965e9 / 1e12
    contraction = contraction_used(args, W.prob, getattr(W, "H", None) or getattr(W, "keep", 1))
    roofline["contraction"] = contraction
    roofline["alu"] = {"bound": "alu", "achieved": flops_per_launch / launch_s / 1e12, "peak": alu_peak,
                       "unit": "TFLOP/s", "frac": flops_per_launch / launch_s / 1e12 / alu_peak,
                       "note": "fp32 FMA lanes: 2*(19*C+120) algorithmic flop per unit-evaluation against "
                               "SMs*128*2*1.965 GHz. With the FFMA2 contraction the kernel is issue/FMA-pipe bound "
                               "(profiles/r1d_photo_config4.md); with the tensor-core contraction the 19*C part runs as "
                               "mma.sync; the L1 data pipe is then the busiest unit (roofline.l1, 75 % under ncu) and the stall "
                               "samples sit on the tap loads (profiles/r1g_photo_config4.md)"}
    per_unit = NCU_PER_UNIT.get((contraction, W.prob["channels"][-1])) if W.prob["dtype"] != "f32" else None
    units_per_launch = W.bytes_per_launch / (4 * W.prob["channels"][-1] * (4 if W.prob["dtype"] == "f32" else 2))
    if per_unit and per_unit["l1_wavefronts"]:
        # the busiest unit (profiles/r1g_photo_config4.md): the LSU data pipe moves one 128-byte wavefront per
        # clock per SM; wavefronts per unit come from the committed ncu capture, the time from this run
        l1_peak = prop.multi_processor_count * 1.965e9
        l1_rate = units_per_launch * per_unit["l1_wavefronts"] / launch_s
        roofline["l1"] = {"bound": "l1-data-pipe", "achieved": l1_rate / 1e9, "peak": l1_peak / 1e9, "unit": "Gwavefront/s",
                          "frac": l1_rate / l1_peak, "wavefronts_per_unit": per_unit["l1_wavefronts"],
                          "algorithmic_wavefronts_per_unit": (4 * W.prob["channels"][-1] * 2 + W.prob["channels"][-1] * 2) / 128.0,
                          "source": per_unit["source"],
                          "note": "l1tex__data_pipe_lsu_wavefronts per unit (global + shared + shuffles + local) x units "
                                  "per launch / launch time against SMs x 1 wavefront/clk x 1.965 GHz; the algorithmic "
                                  "floor is the 4 taps + the reference row (5 x 128 B at C = 64 bf16)"}
    # t_model = max(compulsory HBM bytes / HBM peak, gather bytes / L2 gather peak, flops / FMA
    # peak); the L2 term is filled in below when the probe runs. Instruction issue (warp instructions per unit from
    # the committed ncu captures) is listed beside it because it is the term that binds.
    compulsory = float(map_bytes) / max(1, W.prob["n_levels"])          # one level's map read once per pass
    model = {"t_hbm_compulsory_ms": compulsory / (peak * 1e9) * 1e3, "t_fma_ms": flops_per_launch / (alu_peak * 1e12) * 1e3,
             "t_l2_gather_ms": None, "t_run_ms": launch_s * 1e3}
    if contraction == "mma":
        # the 19*C part is not on the FMA lanes: what stays there is the lift (2*120 flop per unit); the Gram runs as
        # C/16 k-steps x 2 HMMA.16816 per 4 units (4096 flop each, a quarter of it useful) against the mma.sync rate
        # measured on this pool's B200 (550 TFLOP/s dense-equivalent)
        C_last = W.prob["channels"][-1]
        model["t_fma_ms"] = units_per_launch * 2 * 120 / (alu_peak * 1e12) * 1e3
        model["t_tensor_ms"] = units_per_launch * (C_last / 16.0) * 2 * 4096 / 4 / 550e12 * 1e3
        model["fma_note"] = "mma contraction: t_fma_ms = lift only (2*120 flop per unit); t_tensor_ms = issued mma.sync flop / 550 TFLOP/s"
    if per_unit:
        model["t_issue_ms"] = units_per_launch * per_unit["inst"] / (prop.multi_processor_count * 4 * 1.965e9) * 1e3
        model["issue_source"] = "warp instructions per unit from " + per_unit["source"]
        if per_unit["l1_wavefronts"]:
            model["t_l1_pipe_ms"] = units_per_launch * per_unit["l1_wavefronts"] / (prop.multi_processor_count * 1.965e9) * 1e3
    roofline["model"] = model
    if rank == 0 and not args.no_probe:
        # the build's own micro-benchmark: random gathers with the kernel's access shape
        tap = 4 * W.prob["channels"][-1] * (4 if W.prob["dtype"] == "f32" else 2) // 4      # one tap = one pixel
        tap = 1 << (tap.bit_length() - 1)
        l2g = binding.probe_gather(16 << 20, tap, 5, local_rank)
        hbmg = binding.probe_gather(4 << 30, tap, 5, local_rank)
        roofline["gather_peaks"] = {"vec_bytes": tap, "l2_resident_16MiB_gbs": l2g, "hbm_4GiB_gbs": hbmg,
                                    "frac_of_l2_gather_peak": achieved / l2g if l2g else None,
                                    "frac_of_hbm_gather_peak": achieved / hbmg if hbmg else None,
                                    "source": "pilot_refine_probe_gather, measured in this run"}
        model["t_l2_gather_ms"] = W.bytes_per_launch / (l2g * 1e9) * 1e3 if l2g else None
    terms = {k: v for k, v in model.items() if k.startswith("t_") and k != "t_run_ms" and v}
    model["binds"] = max(terms, key=terms.get)
    model["t_model_over_t_run"] = max(terms.values()) / model["t_run_ms"]

    # ---- end to end through the C-ABI with HOST buffers: H2D of every input + D2H of the outputs per step
    e2e = None
    if not args.no_e2e:
        n_e2e = max(1, min(args.steps, 10))
        barrier()
        dt, h2d, d2h = W.e2e(stream, n_e2e)
        n_e2e = getattr(W, "e2e_steps", n_e2e)
        tt = torch.tensor([dt], dtype=torch.float64, device=f"cuda:{local_rank}")
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e = {"value": world * units * n_e2e / float(tt.item()), "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": n_e2e}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        cp = W.cpu_problem()
        v, desc, threads = oracle_sample(cp, cores) if cp is not None else W.cpu_time(cores)
        cpu = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc}

    if rank == 0:
        cfg = {"workload": args.config, "exec_mode": args.mode, "math_mode": args.math}
        cfg.update(W.config())
        cfg.update({"map_bytes": map_bytes, "l2_bytes": int(l2_bytes),
                    "l2_policy": "L2 flushed between timed steps" if need_flush else "inputs larger than L2",
                    "sharding": "hypotheses across ranks, no data-path collective; one 13-float-per-hypothesis "
                                "all-gather + arg-min ends the step when n_gpus > 1"})
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None,
                "dtype": "f32" if contraction == "fp32" else W.prob["dtype"] + " mma.sync products, f32 accumulate; f32 elsewhere",
                "data": "synthetic", "config": cfg,
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
                "gpu_launches": int(launches_per_step * args.steps), "clocks": sampler.summary()}
        print(json.dumps(line))
    W.close()
    if use_dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

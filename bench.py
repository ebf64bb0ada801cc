#!/usr/bin/env python
"""bench.py — point-hypothesis LM iterations per second of pilot_refine_run on B200 (BASELINE.json metric).

A step is one pass of the whole hot path (all levels, all LM iterations, priors, solves)
over one batch of synthetic input. Default workload: config 4 (the configuration north_star's target is quoted
on; 265 MB map > L2). `--impl reference` times the CPU oracle on the host cores instead.
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

# dram__bytes_read.sum + dram__bytes_write.sum per photo_pass_kernel launch from the committed ncu --set full
# capture of this command (profiles/); None until a capture for that workload exists.
NCU_TRAFFIC_BYTES = {}


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


def make_problem(name, rank):
    from paper_2606_31098_b200 import workloads as wl
    prob = wl.make(name)
    if rank:  # weak scaling: every rank refines its own shard of hypotheses around the same scene
        rng = np.random.Generator(np.random.PCG64(wl.BASE_SEED + 1000 * rank))
        T = prob["gt_pose"].reshape(3, 4)
        rot, tr = (10.0, 20.0) if name == "config2" else (5.0, 10.0)
        prob["init_poses"] = wl.perturbed_poses(rng, T, prob["init_poses"].shape[0], rot, tr, first_is_gt=False)
    return prob


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


def run_reference(args, rank):
    if rank != 0:
        return
    prob = make_problem(args.config, 0)
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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="config4", choices=["config1", "config2", "config4"])
    ap.add_argument("--chunk", type=int, default=0, help="anchors per CTA (0 = heuristic)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
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
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    prob = make_problem(args.config, rank)
    params = prob["params"]
    di = binding.DeviceInputs(prob, local_rank)
    ref = binding.Refiner.for_inputs(di, params, local_rank)
    if args.chunk:
        ref.set_chunk(args.chunk)
    stream = torch.cuda.current_stream(local_rank)
    map_bytes = sum(int(np.asarray(q).nbytes) for q in prob["query_feat"])
    l2_bytes = torch.cuda.get_device_properties(local_rank).L2_cache_size
    need_flush = map_bytes <= l2_bytes
    flush = torch.empty(max(2 * l2_bytes, 1 << 28), dtype=torch.uint8, device=f"cuda:{local_rank}") if need_flush else None
    light = ("poses", "cost", "n_valid", "status", "iter_hessian", "iter_gradient", "iter_cost", "iter_lambda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(local_rank)

    for _ in range(max(3, args.warmup)):
        out = ref.run(di, params, stream, light)
    barrier()
    launches_per_step = ref.last_launches
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    for s, e in ev:
        if flush is not None:
            flush.fill_(1)                 # evict the map from L2 between timed steps (outside the events)
        s.record(stream)
        out = ref.run(di, params, stream, light)
        e.record(stream)
    barrier()
    sampler.stop_flag = True
    sampler.join()
    total_ms = sum(s.elapsed_time(e) for s, e in ev)
    t = torch.tensor([total_ms], dtype=torch.float64, device=f"cuda:{local_rank}")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms = float(t.item())
    units = prob["units"]
    value = world * units * args.steps / (total_ms * 1e-3)
    cost = out["cost"].cpu().numpy()
    assert np.isfinite(cost).any(), "no hypothesis ended with a finite cost"

    # ---- roofline of the dominant kernel (photo_pass_kernel): algorithmic gather bytes per launch / launch time
    H, L = prob["init_poses"].shape[0], prob["n_levels"]
    es = 4 if prob["dtype"] == "f32" else 2
    pass_launches = sum(k + 1 for k in params["iters"])
    bytes_per_launch = float(np.mean([H * prob["points"][l].shape[0] * 4 * prob["channels"][l] * es
                                      for l in range(L) for _ in range(params["iters"][l] + 1)]))
    launch_s = (total_ms * 1e-3 / args.steps) / pass_launches   # init kernel + gaps included: conservative
    peak, peak_src = load_peaks()
    achieved = bytes_per_launch / launch_s / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": NCU_TRAFFIC_BYTES.get(args.config), "kernel": "photo_pass_kernel",
                "algorithmic_bytes_per_launch": bytes_per_launch, "launch_ms": launch_s * 1e3,
                "peak_source": peak_src,
                "note": "4*C*s gather bytes per (anchor,hypothesis) unit x H*N units per launch; taps are served "
                        "through L2, so achieved may exceed the HBM copy peak when L2 reuse is high"}

    # ---- end to end through the C-ABI with HOST buffers (pinned): H2D of every input + D2H of every output per step
    e2e = None
    if not args.no_e2e:
        hi = binding.DeviceInputs(prob, local_rank, host=True)
        href = binding.Refiner.for_inputs(hi, params, local_rank, host_path=True)
        if args.chunk:
            href.set_chunk(args.chunk)
        T = sum(params["iters"])
        d2h = H * (48 + 4 + 4 + 4) + T * H * (144 + 24 + 4 + 4)
        n_e2e = max(1, min(args.steps, 5))
        href.run(hi, params, stream, light)
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            href.run(hi, params, stream, light)     # synchronises the stream before returning
        torch.cuda.synchronize(local_rank)
        dt = time.perf_counter() - t0
        tt = torch.tensor([dt], dtype=torch.float64, device=f"cuda:{local_rank}")
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e = {"value": world * units * n_e2e / float(tt.item()), "unit": UNIT,
               "h2d_bytes_per_step": int(hi.h2d_bytes), "d2h_bytes_per_step": int(d2h), "steps": n_e2e}
        href.close()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, desc, threads = oracle_sample(prob, os.cpu_count() or 1)
        cpu = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(3, args.warmup), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": args.config, "hypotheses_per_gpu": H,
                           "points": [int(p.shape[0]) for p in prob["points"]], "channels": prob["channels"],
                           "feat_dtype": prob["dtype"], "iters": params["iters"], "levels": L,
                           "map_bytes": map_bytes, "l2_bytes": int(l2_bytes),
                           "l2_policy": "L2 flushed between timed steps" if need_flush else "inputs larger than L2",
                           "sharding": "hypotheses across ranks, no data-path collective"},
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
                "gpu_launches": int(launches_per_step * args.steps), "clocks": sampler.summary()}
        print(json.dumps(line))
    ref.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

"""Thin Python binding of include/pilot_refine.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of csrc/pilot_refine.cu; torch is used for device
memory and streams. There is NO CPU fallback: if the CUDA library is missing or no GPU is present
the calls raise. This module never imports the oracle.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

MAX_LEVELS = 4
DTYPE_CODE = {"f32": 0, "bf16": 1, "f16": 2}
LOSS_CODE = {"l2": 0, "huber": 1, "cauchy": 2}
RANGE_CODE = {"off": 0, "height": 1, "march": 2}
LM_CODE = {"adaptive": 0, "fixed": 1}
DAMP_CODE = {"identity": 0, "diag": 1}
GRAD_CODE = {"bilinear_exact": 0, "central_sampled": 1}
ERRORS = {-1: "bad argument", -2: "workspace too small", -3: "unsupported shape / mode", -4: "CUDA error"}

EXPORTS = ["pilot_refine_workspace_bytes", "pilot_refine_create", "pilot_refine_run", "pilot_refine_destroy",
           "pilot_refine_create_host", "pilot_refine_run_host", "pilot_refine_last_launches"]


class Config(C.Structure):
    _fields_ = [("device", C.c_int), ("n_levels", C.c_int),
                ("width", C.c_int * MAX_LEVELS), ("height", C.c_int * MAX_LEVELS),
                ("channels", C.c_int * MAX_LEVELS), ("feat_dtype", C.c_int),
                ("max_hypotheses", C.c_int), ("max_points", C.c_int), ("max_total_iters", C.c_int),
                ("workspace_dev", C.c_void_p), ("workspace_bytes", C.c_size_t)]


class Inputs(C.Structure):
    _fields_ = [("n_hypotheses", C.c_int), ("n_points", C.c_int * MAX_LEVELS),
                ("query_feat_dev", C.c_void_p * MAX_LEVELS), ("query_conf_dev", C.c_void_p * MAX_LEVELS),
                ("intrinsics", (C.c_float * 4) * MAX_LEVELS),
                ("points_dev", C.c_void_p * MAX_LEVELS), ("ref_feat_dev", C.c_void_p * MAX_LEVELS),
                ("init_poses_dev", C.c_void_p),
                ("gravity_world", C.c_float * 3), ("gravity_imu", C.c_float * 3),
                ("range_ray_cam", C.c_float * 3), ("range_meas", C.c_float),
                ("dsm_dev", C.c_void_p), ("dsm_width", C.c_int), ("dsm_height", C.c_int),
                ("dsm_origin_x", C.c_float), ("dsm_origin_y", C.c_float), ("dsm_gsd", C.c_float)]


class Params(C.Structure):
    _fields_ = [("iters", C.c_int * MAX_LEVELS), ("loss", C.c_int), ("loss_scale", C.c_float),
                ("lm_mode", C.c_int), ("damp_mode", C.c_int),
                ("lambda_init", C.c_float), ("lambda_up", C.c_float), ("lambda_down", C.c_float),
                ("lambda_min", C.c_float), ("lambda_max", C.c_float),
                ("grad_mode", C.c_int), ("z_near", C.c_float), ("min_valid", C.c_int),
                ("w_gravity", C.c_float), ("gravity_scale", C.c_float),
                ("range_mode", C.c_int), ("w_range", C.c_float), ("range_scale", C.c_float),
                ("march_steps", C.c_int), ("bisect_steps", C.c_int), ("march_tfar_scale", C.c_float)]


class Outputs(C.Structure):
    _fields_ = [("poses_dev", C.c_void_p), ("cost_dev", C.c_void_p), ("n_valid_dev", C.c_void_p),
                ("status_dev", C.c_void_p), ("iter_hessian_dev", C.c_void_p),
                ("iter_gradient_dev", C.c_void_p), ("iter_cost_dev", C.c_void_p),
                ("iter_lambda_dev", C.c_void_p)]


DEFAULT_PARAMS = dict(
    iters=[10], loss="huber", loss_scale=0.1, lm_mode="adaptive", damp_mode="identity",
    lambda_init=1e-2, lambda_up=10.0, lambda_down=0.1, lambda_min=1e-8, lambda_max=1e8,
    grad_mode="bilinear_exact", z_near=0.1, min_valid=8,
    w_gravity=0.0, gravity_scale=0.1, range_mode="off", w_range=1.0, range_scale=5.0,
    march_steps=64, bisect_steps=8, march_tfar_scale=2.0)

_lib = None


def lib():
    """Load csrc/libpilot_refine.so. Raises if it is absent: the product has no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(_build.LIB):
            raise RuntimeError(f"{_build.LIB} is missing: run `python -m paper_2606_31098_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(_build.LIB)
        L.pilot_refine_workspace_bytes.argtypes = [C.POINTER(Config)]
        L.pilot_refine_workspace_bytes.restype = C.c_size_t
        L.pilot_refine_create.argtypes = [C.POINTER(Config), C.POINTER(C.c_void_p)]
        L.pilot_refine_create.restype = C.c_int
        L.pilot_refine_create_host.argtypes = [C.POINTER(Config), C.c_int, C.c_int, C.POINTER(C.c_void_p)]
        L.pilot_refine_create_host.restype = C.c_int
        for name in ("pilot_refine_run", "pilot_refine_run_host"):
            fn = getattr(L, name)
            fn.argtypes = [C.c_void_p, C.POINTER(Inputs), C.POINTER(Params), C.POINTER(Outputs), C.c_void_p]
            fn.restype = C.c_int
        L.pilot_refine_destroy.argtypes = [C.c_void_p]
        L.pilot_refine_destroy.restype = C.c_int
        L.pilot_refine_last_launches.argtypes = [C.c_void_p]
        L.pilot_refine_last_launches.restype = C.c_int
        L.pilot_refine_set_chunk.argtypes = [C.c_void_p, C.c_int]
        L.pilot_refine_set_chunk.restype = C.c_int
        _lib = L
    return _lib


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"{what} failed: {rc} ({ERRORS.get(rc, '?')})")


def make_params(P_in, n_levels):
    P = dict(DEFAULT_PARAMS)
    P.update(P_in or {})
    assert len(P["iters"]) == n_levels, "params.iters needs one entry per level"
    par = Params()
    for l in range(n_levels):
        par.iters[l] = int(P["iters"][l])
    par.loss, par.loss_scale = LOSS_CODE[P["loss"]], P["loss_scale"]
    par.lm_mode, par.damp_mode = LM_CODE[P["lm_mode"]], DAMP_CODE[P["damp_mode"]]
    par.lambda_init, par.lambda_up, par.lambda_down = P["lambda_init"], P["lambda_up"], P["lambda_down"]
    par.lambda_min, par.lambda_max = P["lambda_min"], P["lambda_max"]
    par.grad_mode, par.z_near, par.min_valid = GRAD_CODE[P["grad_mode"]], P["z_near"], int(P["min_valid"])
    par.w_gravity, par.gravity_scale = P["w_gravity"], P["gravity_scale"]
    par.range_mode, par.w_range, par.range_scale = RANGE_CODE[P["range_mode"]], P["w_range"], P["range_scale"]
    par.march_steps, par.bisect_steps = int(P["march_steps"]), int(P["bisect_steps"])
    par.march_tfar_scale = P["march_tfar_scale"]
    return par, P


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("pilot_refine needs a CUDA device (sm_100a); there is no CPU fallback")
    return torch


def _as_bytes_tensor(torch, a, device, pin=False):
    """numpy array (any dtype, incl. uint16 bf16 bit patterns) -> torch uint8 tensor with the same bytes."""
    a = np.ascontiguousarray(a)
    t = torch.from_numpy(a.view(np.uint8).reshape(-1))
    if device is not None:
        return t.to(device)
    return t.pin_memory() if pin else t


class DeviceInputs:
    """A problem dict (paper_2606_31098_b200.workloads) resident in HBM as torch tensors + the Inputs struct."""

    def __init__(self, prob, device=0, host=False):
        torch = _torch()
        dev = None if host else torch.device("cuda", device)
        self.keep = []
        L = int(prob["n_levels"])
        self.n_levels, self.dtype = L, prob["dtype"]
        self.width, self.height = [int(v) for v in prob["width"]], [int(v) for v in prob["height"]]
        self.channels = [int(v) for v in prob["channels"]]
        inp = Inputs()
        self.h2d_bytes = 0

        def put(a, dt=None):
            a = np.ascontiguousarray(a if dt is None else np.asarray(a, dtype=dt))
            t = _as_bytes_tensor(torch, a, dev, pin=host)
            self.keep.append(t)
            self.h2d_bytes += t.numel()
            return t.data_ptr() if t.numel() else None

        self.n_hyp = int(prob["init_poses"].shape[0])
        inp.n_hypotheses = self.n_hyp
        for l in range(L):
            inp.query_feat_dev[l] = put(prob["query_feat"][l])
            qc = prob.get("query_conf", [None] * L)[l]
            inp.query_conf_dev[l] = None if qc is None else put(qc, np.float32)
            for k in range(4):
                inp.intrinsics[l][k] = float(prob["intrinsics"][l][k])
            pts = np.asarray(prob["points"][l], np.float32)
            inp.n_points[l] = pts.shape[0]
            inp.points_dev[l] = put(pts)
            inp.ref_feat_dev[l] = put(prob["ref_feat"][l])
        inp.init_poses_dev = put(prob["init_poses"], np.float32)
        for k in range(3):
            inp.gravity_world[k] = float(prob["gravity_world"][k])
            inp.gravity_imu[k] = float(prob["gravity_imu"][k])
            inp.range_ray_cam[k] = float(prob["range_ray_cam"][k])
        inp.range_meas = float(prob["range_meas"])
        dsm = prob.get("dsm")
        if dsm is not None:
            inp.dsm_dev = put(dsm, np.float32)
            inp.dsm_height, inp.dsm_width = dsm.shape
        inp.dsm_origin_x, inp.dsm_origin_y = float(prob["dsm_origin"][0]), float(prob["dsm_origin"][1])
        inp.dsm_gsd = float(prob["dsm_gsd"])
        self.inp = inp
        self.max_points = max(int(inp.n_points[l]) for l in range(L))


class Refiner:
    """Owns one pilot_refine handle and its output tensors. run() is asynchronous on the given stream."""

    def __init__(self, n_levels, width, height, channels, dtype, max_hypotheses, max_points, max_total_iters,
                 device=0, host_path=False, max_dsm=(0, 0)):
        torch = _torch()
        self.torch, self.device = torch, device
        cfg = Config()
        cfg.device, cfg.n_levels, cfg.feat_dtype = device, n_levels, DTYPE_CODE[dtype]
        for l in range(n_levels):
            cfg.width[l], cfg.height[l], cfg.channels[l] = int(width[l]), int(height[l]), int(channels[l])
        cfg.max_hypotheses, cfg.max_points, cfg.max_total_iters = int(max_hypotheses), int(max_points), int(max_total_iters)
        self.cfg, self.host_path = cfg, host_path
        self.handle = C.c_void_p()
        L = lib()
        if host_path:
            _check(L.pilot_refine_create_host(C.byref(cfg), int(max_dsm[0]), int(max_dsm[1]), C.byref(self.handle)),
                   "pilot_refine_create_host")
        else:
            nbytes = L.pilot_refine_workspace_bytes(C.byref(cfg))
            if nbytes == 0:
                raise RuntimeError("pilot_refine_workspace_bytes: bad config")
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=torch.device("cuda", device))
            base = (self.workspace.data_ptr() + 255) // 256 * 256
            cfg.workspace_dev, cfg.workspace_bytes = base, nbytes
            _check(L.pilot_refine_create(C.byref(cfg), C.byref(self.handle)), "pilot_refine_create")
        H, T = int(max_hypotheses), max(1, int(max_total_iters))
        kw = dict(device=torch.device("cuda", device)) if not host_path else dict(pin_memory=True)
        self.o = dict(poses=torch.zeros(H, 12, dtype=torch.float32, **kw), cost=torch.zeros(H, dtype=torch.float32, **kw),
                      n_valid=torch.zeros(H, dtype=torch.int32, **kw), status=torch.zeros(H, dtype=torch.int32, **kw),
                      iter_hessian=torch.zeros(T * H * 36, dtype=torch.float32, **kw),
                      iter_gradient=torch.zeros(T * H * 6, dtype=torch.float32, **kw),
                      iter_cost=torch.zeros(T * H, dtype=torch.float32, **kw),
                      iter_lambda=torch.zeros(T * H, dtype=torch.float32, **kw))

    @classmethod
    def for_inputs(cls, di, params, device=0, host_path=False):
        P = dict(DEFAULT_PARAMS); P.update(params or {})
        dsm = (int(di.inp.dsm_width), int(di.inp.dsm_height))
        return cls(di.n_levels, di.width, di.height, di.channels, di.dtype, max(1, di.n_hyp), max(1, di.max_points),
                   sum(P["iters"]), device=device, host_path=host_path, max_dsm=dsm)

    def set_chunk(self, chunk):
        _check(lib().pilot_refine_set_chunk(self.handle, int(chunk)), "pilot_refine_set_chunk")

    def run(self, di, params, stream=None, outputs=("poses", "cost", "n_valid", "status", "iter_hessian",
                                                    "iter_gradient", "iter_cost", "iter_lambda")):
        """Enqueue one refinement. Returns dict of output tensors (views; valid once the stream reaches them)."""
        torch = self.torch
        par, P = make_params(params, di.n_levels)
        out = Outputs()
        for name in outputs:
            setattr(out, name + "_dev", self.o[name].data_ptr())
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        fn = lib().pilot_refine_run_host if self.host_path else lib().pilot_refine_run
        _check(fn(self.handle, C.byref(di.inp), C.byref(par), C.byref(out), C.c_void_p(stream.cuda_stream)),
               "pilot_refine_run_host" if self.host_path else "pilot_refine_run")
        H, T = di.n_hyp, sum(P["iters"])
        res = {}
        for name in outputs:
            t = self.o[name]
            if name == "iter_hessian": t = t[:T * H * 36].view(T, H, 36)
            elif name == "iter_gradient": t = t[:T * H * 6].view(T, H, 6)
            elif name in ("iter_cost", "iter_lambda"): t = t[:T * H].view(T, H)
            else: t = t[:H]
            res[name] = t
        return res

    @property
    def last_launches(self):
        return lib().pilot_refine_last_launches(self.handle)

    def close(self):
        if self.handle:
            lib().pilot_refine_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def refine(prob, params=None, device=0):
    """One-shot convenience: upload a problem dict, run, synchronise, return numpy outputs."""
    torch = _torch()
    di = DeviceInputs(prob, device)
    P = dict(prob.get("params", {})); P.update(params or {})
    r = Refiner.for_inputs(di, P, device)
    out = r.run(di, P)
    torch.cuda.synchronize(device)
    res = {k: v.cpu().numpy() for k, v in out.items()}
    res["status"] = res["status"].view(np.uint32)
    res["launches"] = r.last_launches
    r.close()
    return res

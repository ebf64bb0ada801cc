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

SEED_CODE = {"camera": 0, "world": 1}
EXEC_CODE = {"auto": 0, "passes": 1, "resident": 2, "split": 3}
MATH_CODE = {"auto": 0, "fp32": 1, "mma": 2}
TOPK_MAX = 8192

EXPORTS = ["pilot_refine_workspace_bytes", "pilot_refine_create", "pilot_refine_run", "pilot_refine_destroy",
           "pilot_refine_create_host", "pilot_refine_run_host", "pilot_refine_submit_host",
           "pilot_refine_wait_host", "pilot_refine_last_launches",
           "pilot_refine_run_levels", "pilot_refine_set_exec_mode", "pilot_refine_set_math_mode", "pilot_refine_grid_offsets", "pilot_refine_seed_hypotheses",
           "pilot_refine_select_best", "pilot_refine_prune_topk",
           "pilot_refine_sequence_create", "pilot_refine_sequence_set_prior", "pilot_refine_sequence_upload",
           "pilot_refine_sequence_step", "pilot_refine_sequence_results", "pilot_refine_sequence_last_frame",
           "pilot_refine_sequence_last_launches", "pilot_refine_sequence_destroy", "pilot_refine_probe_gather",
           "pilot_refine_probe_unit_gather", "pilot_refine_last_visible_evals", "pilot_refine_last_plan",
           "pilot_refine_set_iterate_outputs", "pilot_refine_unrolled_backward", "pilot_refine_unrolled_backward_scratch_bytes",
           "pilot_refine_sort_anchors", "pilot_refine_sort_anchors_temp_bytes",
           "pilot_refine_set_grid_host", "pilot_refine_submit_pruned_host",
           "pilot_refine_reprojection_loss_grad", "pilot_refine_lm_step_adjoint", "pilot_refine_photo_backward",
           "pilot_refine_footprint", "pilot_refine_lift_anchors", "pilot_refine_reprojection_loss",
           "pilot_refine_run_static", "pilot_refine_static_workspace_bytes"]
SEQ_ROW = 16


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


class UnrolledRecords(C.Structure):
    _fields_ = [("iter_hessian_dev", C.c_void_p), ("iter_gradient_dev", C.c_void_p), ("iter_lambda_dev", C.c_void_p),
                ("iter_poses_dev", C.c_void_p), ("iter_accept_dev", C.c_void_p), ("final_poses_dev", C.c_void_p)]


class Supervision(C.Structure):
    _fields_ = [("pose_star", C.c_float * 12), ("points_dev", C.c_void_p), ("n_points", C.c_int),
                ("intrinsics", C.c_float * 4), ("width", C.c_int), ("height", C.c_int),
                ("alpha", C.c_float), ("scale", C.c_float), ("step_weights", C.POINTER(C.c_float))]


class UnrolledGrads(C.Structure):
    _fields_ = [("grad_feat_dev", C.c_void_p * MAX_LEVELS), ("grad_ref_dev", C.c_void_p * MAX_LEVELS),
                ("grad_conf_dev", C.c_void_p * MAX_LEVELS), ("grad_init_pose_dev", C.c_void_p), ("loss_dev", C.c_void_p)]


class SequenceConfig(C.Structure):
    _fields_ = [("n_hypotheses", C.c_int), ("offsets", C.c_void_p), ("seed_frame", C.c_int),
                ("dsm", C.c_void_p), ("dsm_width", C.c_int), ("dsm_height", C.c_int),
                ("dsm_origin_x", C.c_float), ("dsm_origin_y", C.c_float), ("dsm_gsd", C.c_float),
                ("gravity_world", C.c_float * 3), ("max_frames", C.c_int)]


class Frame(C.Structure):
    _fields_ = [("n_points", C.c_int * MAX_LEVELS),
                ("query_feat", C.c_void_p * MAX_LEVELS), ("query_conf", C.c_void_p * MAX_LEVELS),
                ("points", C.c_void_p * MAX_LEVELS), ("ref_feat", C.c_void_p * MAX_LEVELS),
                ("intrinsics", (C.c_float * 4) * MAX_LEVELS),
                ("gravity_imu", C.c_float * 3), ("range_ray_cam", C.c_float * 3), ("range_meas", C.c_float),
                ("arrays_pinned", C.c_int)]


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
        L.pilot_refine_wait_host.argtypes = [C.c_void_p]
        L.pilot_refine_wait_host.restype = C.c_int
        for name in ("pilot_refine_run", "pilot_refine_run_host", "pilot_refine_submit_host"):
            fn = getattr(L, name)
            fn.argtypes = [C.c_void_p, C.POINTER(Inputs), C.POINTER(Params), C.POINTER(Outputs), C.c_void_p]
            fn.restype = C.c_int
        L.pilot_refine_destroy.argtypes = [C.c_void_p]
        L.pilot_refine_destroy.restype = C.c_int
        L.pilot_refine_run_static.argtypes = [C.POINTER(Config), C.POINTER(Inputs), C.POINTER(Params), C.POINTER(Outputs),
                                              C.c_void_p, C.POINTER(C.c_int)]
        L.pilot_refine_run_static.restype = C.c_int
        L.pilot_refine_static_workspace_bytes.argtypes = []
        L.pilot_refine_static_workspace_bytes.restype = C.c_size_t
        L.pilot_refine_last_launches.argtypes = [C.c_void_p]
        L.pilot_refine_last_launches.restype = C.c_int
        L.pilot_refine_set_chunk.argtypes = [C.c_void_p, C.c_int]
        L.pilot_refine_set_chunk.restype = C.c_int
        L.pilot_refine_set_exec_mode.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.pilot_refine_set_exec_mode.restype = C.c_int
        L.pilot_refine_set_math_mode.argtypes = [C.c_void_p, C.c_int]
        L.pilot_refine_set_math_mode.restype = C.c_int
        L.pilot_refine_run_levels.argtypes = [C.c_void_p, C.POINTER(Inputs), C.POINTER(Params), C.POINTER(Outputs),
                                              C.c_int, C.c_int, C.c_void_p]
        L.pilot_refine_run_levels.restype = C.c_int
        L.pilot_refine_grid_offsets.argtypes = [C.c_float, C.c_float, C.POINTER(C.c_float), C.c_int,
                                                C.POINTER(C.c_float), C.POINTER(C.c_float), C.c_int]
        L.pilot_refine_grid_offsets.restype = C.c_int
        L.pilot_refine_seed_hypotheses.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.pilot_refine_seed_hypotheses.restype = C.c_int
        L.pilot_refine_select_best.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                               C.c_void_p]
        L.pilot_refine_select_best.restype = C.c_int
        L.pilot_refine_prune_topk.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p,
                                              C.c_void_p, C.c_void_p]
        L.pilot_refine_prune_topk.restype = C.c_int
        L.pilot_refine_sequence_create.argtypes = [C.POINTER(Config), C.POINTER(SequenceConfig), C.POINTER(C.c_void_p)]
        L.pilot_refine_sequence_set_prior.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.pilot_refine_sequence_upload.argtypes = [C.c_void_p, C.POINTER(Frame)]
        L.pilot_refine_sequence_step.argtypes = [C.c_void_p, C.POINTER(Params), C.c_void_p]
        L.pilot_refine_sequence_results.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.pilot_refine_sequence_last_frame.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.pilot_refine_sequence_last_launches.argtypes = [C.c_void_p]
        L.pilot_refine_sequence_destroy.argtypes = [C.c_void_p]
        L.pilot_refine_footprint.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.c_int, C.c_int, C.c_void_p, C.c_int, C.c_int,
                                             C.c_float, C.c_float, C.c_float, C.c_int, C.c_float, C.c_void_p, C.c_void_p]
        L.pilot_refine_footprint.restype = C.c_int
        L.pilot_refine_lift_anchors.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_int,
                                                C.c_float, C.c_float, C.c_float, C.c_void_p, C.c_void_p]
        L.pilot_refine_lift_anchors.restype = C.c_int
        L.pilot_refine_reprojection_loss.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_float), C.c_void_p, C.c_int,
                                                     C.POINTER(C.c_float), C.c_int, C.c_int, C.c_float, C.c_float, C.c_float,
                                                     C.c_void_p, C.c_void_p, C.c_void_p]
        L.pilot_refine_reprojection_loss.restype = C.c_int
        L.pilot_refine_probe_gather.argtypes = [C.c_int, C.c_size_t, C.c_int, C.c_int, C.POINTER(C.c_double)]
        L.pilot_refine_probe_gather.restype = C.c_int
        L.pilot_refine_probe_unit_gather.argtypes = [C.c_int, C.c_size_t, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_double)]
        L.pilot_refine_probe_unit_gather.restype = C.c_int
        L.pilot_refine_last_visible_evals.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_ulonglong)]
        L.pilot_refine_last_visible_evals.restype = C.c_int
        L.pilot_refine_last_plan.argtypes = [C.c_void_p, C.POINTER(C.c_uint), C.POINTER(C.c_uint)]
        L.pilot_refine_last_plan.restype = C.c_int
        L.pilot_refine_sort_anchors_temp_bytes.argtypes = [C.c_int]
        L.pilot_refine_sort_anchors_temp_bytes.restype = C.c_size_t
        L.pilot_refine_sort_anchors.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p,
                                                C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        L.pilot_refine_sort_anchors.restype = C.c_int
        L.pilot_refine_reprojection_loss_grad.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_float), C.c_void_p, C.c_int,
                                                          C.POINTER(C.c_float), C.c_int, C.c_int, C.c_float, C.c_float, C.c_float,
                                                          C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.pilot_refine_reprojection_loss_grad.restype = C.c_int
        L.pilot_refine_lm_step_adjoint.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p,
                                                   C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.pilot_refine_lm_step_adjoint.restype = C.c_int
        L.pilot_refine_photo_backward.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float),
                                                  C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int,
                                                  C.c_int, C.c_float, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                                  C.c_void_p]
        L.pilot_refine_photo_backward.restype = C.c_int
        L.pilot_refine_set_iterate_outputs.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.pilot_refine_set_iterate_outputs.restype = C.c_int
        L.pilot_refine_unrolled_backward_scratch_bytes.argtypes = [C.c_int, C.c_int]
        L.pilot_refine_unrolled_backward_scratch_bytes.restype = C.c_size_t
        L.pilot_refine_unrolled_backward.argtypes = [C.POINTER(Config), C.POINTER(Inputs), C.POINTER(Params), C.POINTER(UnrolledRecords),
                                                     C.POINTER(Supervision), C.POINTER(UnrolledGrads), C.c_void_p, C.c_size_t, C.c_void_p]
        L.pilot_refine_unrolled_backward.restype = C.c_int
        L.pilot_refine_set_grid_host.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.pilot_refine_set_grid_host.restype = C.c_int
        L.pilot_refine_submit_pruned_host.argtypes = [C.c_void_p, C.POINTER(Inputs), C.POINTER(Params), C.c_void_p, C.c_int,
                                                      C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.pilot_refine_submit_pruned_host.restype = C.c_int
        for name in EXPORTS:
            if name.startswith("pilot_refine_sequence_"):
                getattr(L, name).restype = C.c_int
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

        has_poses = prob.get("init_poses") is not None
        self.n_hyp = int(prob["init_poses"].shape[0]) if has_poses else 0
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
        inp.init_poses_dev = put(prob["init_poses"], np.float32) if has_poses else None
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

    def sort_anchors(self, stream=None):
        """Put every level's anchors and reference rows in Morton order on the device (pilot_refine_sort_anchors) and
        point the Inputs struct at the sorted copies. Returns the permutations (cuda int32 tensors, one per level)."""
        torch = _torch()
        perms = []
        for l in range(self.n_levels):
            n = int(self.inp.n_points[l])
            if n == 0:
                perms.append(None)
                continue
            dev = torch.device("cuda", torch.cuda.current_device())
            row = self.channels[l] * (4 if self.dtype == "f32" else 2)
            pts = torch.empty(n * 16, dtype=torch.uint8, device=dev)
            ref = torch.empty(n * row, dtype=torch.uint8, device=dev)
            perm = torch.empty(n, dtype=torch.int32, device=dev)
            tb = lib().pilot_refine_sort_anchors_temp_bytes(n)
            tmp = torch.empty(tb + 256, dtype=torch.uint8, device=dev)
            tptr = (tmp.data_ptr() + 255) // 256 * 256
            st = stream if stream is not None else torch.cuda.current_stream()
            _check(lib().pilot_refine_sort_anchors(self.inp.points_dev[l], self.inp.ref_feat_dev[l], n, self.channels[l],
                                                   DTYPE_CODE[self.dtype], pts.data_ptr(), ref.data_ptr(), perm.data_ptr(),
                                                   tptr, tb, C.c_void_p(st.cuda_stream)), "pilot_refine_sort_anchors")
            st.synchronize()                      # tmp may go; the sorted buffers are kept alive by self.keep
            self.keep += [pts, ref]
            self.inp.points_dev[l], self.inp.ref_feat_dev[l] = pts.data_ptr(), ref.data_ptr()
            perms.append(perm)
        return perms


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

    # ---- pipelined host path: submit run k+1 before waiting for run k so that its upload overlaps run k's kernels
    def submit(self, di, params, stream=None, outputs=("poses", "cost", "n_valid", "status")):
        assert self.host_path, "submit/wait is the host-buffer path"
        torch = self.torch
        if not hasattr(self, "_sets"):
            self._sets = [self.o, {k: torch.zeros_like(v).pin_memory() for k, v in self.o.items()}]
            self._pending, self._nsub = [], 0
        k = self._nsub                                   # host output sets alternate; at most two runs are in flight
        par, P = make_params(params, di.n_levels)
        out = Outputs()
        o = self._sets[k & 1]
        for name in outputs:
            setattr(out, name + "_dev", o[name].data_ptr())
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        t = lib().pilot_refine_submit_host(self.handle, C.byref(di.inp), C.byref(par), C.byref(out),
                                           C.c_void_p(stream.cuda_stream))
        if t < 0:
            _check(t, "pilot_refine_submit_host")
        self._pending.append((k, o, outputs, di.n_hyp, sum(P["iters"])))
        self._nsub = k + 1
        return t

    def wait(self):
        """Blocks until the oldest submitted run's outputs are in (pinned) host memory; returns them (views)."""
        _check(lib().pilot_refine_wait_host(self.handle), "pilot_refine_wait_host")
        k, o, outputs, H, T = self._pending.pop(0)
        return {name: (o[name][:H] if not name.startswith("iter_") else o[name]) for name in outputs}

    @classmethod
    def for_inputs(cls, di, params, device=0, host_path=False):
        P = dict(DEFAULT_PARAMS); P.update(params or {})
        dsm = (int(di.inp.dsm_width), int(di.inp.dsm_height))
        return cls(di.n_levels, di.width, di.height, di.channels, di.dtype, max(1, di.n_hyp), max(1, di.max_points),
                   sum(P["iters"]), device=device, host_path=host_path, max_dsm=dsm)

    def set_exec_mode(self, mode="auto", cluster=0):
        _check(lib().pilot_refine_set_exec_mode(self.handle, EXEC_CODE[mode], int(cluster)), "pilot_refine_set_exec_mode")

    def set_math_mode(self, math="auto"):
        _check(lib().pilot_refine_set_math_mode(self.handle, MATH_CODE[math]), "pilot_refine_set_math_mode")

    def record_iterates(self, on=True):
        """pilot_refine_set_iterate_outputs: the following runs also write, per solve, the pose the recorded system was built
        at (iter_poses [T, H, 12]) and whether its step was accepted (iter_accept [T, H] int32); run() returns them."""
        torch = self.torch
        if on and "iter_poses" not in self.o:
            H, T = self.o["poses"].shape[0], self.o["iter_cost"].numel() // self.o["poses"].shape[0]
            dev = self.o["poses"].device
            self.o["iter_poses"] = torch.zeros(T * H * 12, dtype=torch.float32, device=dev)
            self.o["iter_accept"] = torch.zeros(T * H, dtype=torch.int32, device=dev)
        self._iterates = bool(on)
        _check(lib().pilot_refine_set_iterate_outputs(self.handle, self.o["iter_poses"].data_ptr() if on else None,
                                                      self.o["iter_accept"].data_ptr() if on else None),
               "pilot_refine_set_iterate_outputs")

    def set_chunk(self, chunk):
        _check(lib().pilot_refine_set_chunk(self.handle, int(chunk)), "pilot_refine_set_chunk")

    def run(self, di, params, stream=None, outputs=("poses", "cost", "n_valid", "status", "iter_hessian",
                                                    "iter_gradient", "iter_cost", "iter_lambda"), levels=None):
        """Enqueue one refinement (of pyramid levels [levels[0], levels[1]) if given). Returns dict of output
        tensors (views; valid once the stream reaches them)."""
        torch = self.torch
        par, P = make_params(params, di.n_levels)
        out = Outputs()
        for name in outputs:
            setattr(out, name + "_dev", self.o[name].data_ptr())
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        if levels is not None:
            assert not self.host_path, "run_levels has no host-buffer variant"
            _check(lib().pilot_refine_run_levels(self.handle, C.byref(di.inp), C.byref(par), C.byref(out),
                                                 int(levels[0]), int(levels[1]), C.c_void_p(stream.cuda_stream)),
                   "pilot_refine_run_levels")
        else:
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
        if getattr(self, "_iterates", False):
            res["iter_poses"] = self.o["iter_poses"][:T * H * 12].view(T, H, 12)
            res["iter_accept"] = self.o["iter_accept"][:T * H].view(T, H)
        return res

    @property
    def last_launches(self):
        return lib().pilot_refine_last_launches(self.handle)

    def last_plan(self):
        """(mma_levels, resident_levels) bit masks of the last run: which levels used the tensor-core contraction / the
        cluster-resident kernel."""
        a, b = C.c_uint(), C.c_uint()
        _check(lib().pilot_refine_last_plan(self.handle, C.byref(a), C.byref(b)), "pilot_refine_last_plan")
        return int(a.value), int(b.value)

    def last_visible_evals(self, stream=None):
        """Visible (anchor, hypothesis) unit evaluations of the last run, all passes and levels (synchronises the stream)."""
        if stream is None:
            stream = self.torch.cuda.current_stream(self.device)
        n = C.c_ulonglong()
        _check(lib().pilot_refine_last_visible_evals(self.handle, C.c_void_p(stream.cuda_stream), C.byref(n)),
               "pilot_refine_last_visible_evals")
        return int(n.value)

    def close(self):
        if self.handle:
            lib().pilot_refine_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def refine(prob, params=None, device=0, mode="auto", cluster=0, math="auto"):
    """One-shot convenience: upload a problem dict, run, synchronise, return numpy outputs."""
    torch = _torch()
    di = DeviceInputs(prob, device)
    P = dict(prob.get("params", {})); P.update(params or {})
    r = Refiner.for_inputs(di, P, device)
    r.set_exec_mode(mode, cluster)
    r.set_math_mode(math)
    out = r.run(di, P)
    torch.cuda.synchronize(device)
    res = {k: v.cpu().numpy() for k, v in out.items()}
    res["status"] = res["status"].view(np.uint32)
    res["launches"] = r.last_launches
    r.close()
    return res


def unrolled_backward(refiner, di, params, run_out, pose_star, sup_points, sup_intrinsics, width, height, alpha, scale,
                      step_weights=None, grad_conf=False, stream=None):
    """pilot_refine_unrolled_backward: the backward pass through every LM step of the run that produced `run_out` (the dict
    Refiner.run returned with record_iterates() on). L = sum_r step_weights[r-1] L_r(pose after r solves); default weights
    1/T (the paper's average over the unrolled steps). Returns dict: grad_feat / grad_ref (/ grad_conf) lists per level
    (cuda fp32 tensors), grad_init_pose [H, 6], loss [H]. Marshalling only."""
    torch = _torch()
    par, P = make_params(params, di.n_levels)
    H, T = di.n_hyp, sum(P["iters"])
    dev = run_out["poses"].device
    rec = UnrolledRecords()
    rec.iter_hessian_dev, rec.iter_gradient_dev = run_out["iter_hessian"].data_ptr(), run_out["iter_gradient"].data_ptr()
    rec.iter_lambda_dev = run_out["iter_lambda"].data_ptr()
    rec.iter_poses_dev, rec.iter_accept_dev = run_out["iter_poses"].data_ptr(), run_out["iter_accept"].data_ptr()
    rec.final_poses_dev = run_out["poses"].data_ptr()
    w = np.full(max(T, 1), 1.0 / max(T, 1), np.float32) if step_weights is None else np.ascontiguousarray(step_weights, np.float32)
    assert w.size >= T
    sup = Supervision()
    for i, v in enumerate(np.asarray(pose_star, np.float32).reshape(-1)):
        sup.pose_star[i] = float(v)
    sup.points_dev, sup.n_points = sup_points.data_ptr(), int(sup_points.shape[0])
    for i in range(4):
        sup.intrinsics[i] = float(sup_intrinsics[i])
    sup.width, sup.height, sup.alpha, sup.scale = int(width), int(height), float(alpha), float(scale)
    sup.step_weights = w.ctypes.data_as(C.POINTER(C.c_float))
    g = UnrolledGrads()
    res = dict(grad_feat=[], grad_ref=[], grad_conf=[])
    for l in range(di.n_levels):
        gf = torch.zeros(di.height[l], di.width[l], di.channels[l], dtype=torch.float32, device=dev)
        gr = torch.zeros(int(di.inp.n_points[l]), di.channels[l], dtype=torch.float32, device=dev)
        gc = torch.zeros(di.height[l], di.width[l], dtype=torch.float32, device=dev) if (grad_conf and di.inp.query_conf_dev[l]) else None
        g.grad_feat_dev[l], g.grad_ref_dev[l] = gf.data_ptr(), gr.data_ptr()
        g.grad_conf_dev[l] = gc.data_ptr() if gc is not None else None
        res["grad_feat"].append(gf); res["grad_ref"].append(gr); res["grad_conf"].append(gc)
    res["grad_init_pose"] = torch.zeros(H, 6, dtype=torch.float32, device=dev)
    res["loss"] = torch.zeros(H, dtype=torch.float32, device=dev)
    g.grad_init_pose_dev, g.loss_dev = res["grad_init_pose"].data_ptr(), res["loss"].data_ptr()
    nb = lib().pilot_refine_unrolled_backward_scratch_bytes(H, T)
    scratch = torch.empty(nb + 256, dtype=torch.uint8, device=dev)
    sptr = (scratch.data_ptr() + 255) // 256 * 256
    st = stream if stream is not None else torch.cuda.current_stream(dev)
    _check(lib().pilot_refine_unrolled_backward(C.byref(refiner.cfg), C.byref(di.inp), C.byref(par), C.byref(rec), C.byref(sup),
                                                C.byref(g), sptr, nb, C.c_void_p(st.cuda_stream)), "pilot_refine_unrolled_backward")
    st.synchronize()                               # scratch and the host weights may go
    return res


def static_workspace_bytes():
    return int(lib().pilot_refine_static_workspace_bytes())


def run_static(di, params, out, max_hypotheses=None, max_points=None, device=0, stream=None):
    """pilot_refine_run_static: the refinement with the library's file-scope workspace, no handle and no allocation in
    the call. `out`: dict name -> caller-owned cuda tensor (poses [H,12] f32, cost [H] f32, n_valid [H] i32, status [H]
    i32, iter_hessian [T,H,36], iter_gradient [T,H,6], iter_cost [T,H], iter_lambda [T,H]); any subset. Returns the
    number of kernels launched. Asynchronous on `stream`; calls must not overlap on the GPU (they share the workspace)."""
    torch = _torch()
    par, P = make_params(params, di.n_levels)
    cfg = Config()
    cfg.device, cfg.n_levels, cfg.feat_dtype = device, di.n_levels, DTYPE_CODE[di.dtype]
    for l in range(di.n_levels):
        cfg.width[l], cfg.height[l], cfg.channels[l] = int(di.width[l]), int(di.height[l]), int(di.channels[l])
    cfg.max_hypotheses = int(max_hypotheses if max_hypotheses is not None else max(1, di.n_hyp))
    cfg.max_points = int(max_points if max_points is not None else max(1, di.max_points))
    cfg.max_total_iters = sum(P["iters"])
    o = Outputs()
    for name, t in out.items():
        assert t.is_cuda and t.is_contiguous()
        setattr(o, name + "_dev", t.data_ptr())
    n = C.c_int(0)
    _check(lib().pilot_refine_run_static(C.byref(cfg), C.byref(di.inp), C.byref(par), C.byref(o),
                                         _stream_ptr(torch, stream, device), C.byref(n)), "pilot_refine_run_static")
    return int(n.value)


# ------------------------------------------------------------------ hypothesis set

def grid_offsets(xy_range, xy_step, yaw_deg, up):
    """The paper's (x, y, psi) grid as [n, 6] float32 (rotation vector rad, translation m); pure host call."""
    yaw = (C.c_float * len(yaw_deg))(*[float(y) for y in yaw_deg])
    upv = (C.c_float * 3)(*[float(v) for v in up])
    n = lib().pilot_refine_grid_offsets(float(xy_range), float(xy_step), yaw, len(yaw_deg), upv, None, 0)
    if n < 0:
        _check(n, "pilot_refine_grid_offsets")
    out = np.zeros((n, 6), np.float32)
    n2 = lib().pilot_refine_grid_offsets(float(xy_range), float(xy_step), yaw, len(yaw_deg), upv,
                                         out.ctypes.data_as(C.POINTER(C.c_float)), n)
    assert n2 == n
    return out


def _stream_ptr(torch, stream, device):
    if stream is None:
        stream = torch.cuda.current_stream(device)
    return C.c_void_p(stream.cuda_stream)


def seed_hypotheses(base_pose, offsets, frame="camera", out=None, stream=None):
    """base_pose: cuda float32 [12]; offsets: cuda float32 [n, 6] -> cuda float32 [n, 12] (asynchronous)."""
    torch = _torch()
    n = int(offsets.shape[0])
    assert base_pose.is_cuda and offsets.is_cuda and base_pose.dtype == offsets.dtype == torch.float32
    assert base_pose.is_contiguous() and offsets.is_contiguous()
    if out is None:
        out = torch.empty(n, 12, dtype=torch.float32, device=offsets.device)
    _check(lib().pilot_refine_seed_hypotheses(base_pose.data_ptr(), offsets.data_ptr(), n, SEED_CODE[frame],
                                              out.data_ptr(), _stream_ptr(torch, stream, offsets.device)),
           "pilot_refine_seed_hypotheses")
    return out


def select_best(cost, poses, stream=None):
    """cost: cuda float32 [n]; poses: cuda float32 [n, 12] -> (idx int32 [1], pose [12], cost [1]) on the device."""
    torch = _torch()
    n = int(cost.shape[0])
    assert cost.is_cuda and cost.dtype == torch.float32 and cost.is_contiguous() and poses.is_contiguous()
    idx = torch.empty(1, dtype=torch.int32, device=cost.device)
    pose = torch.empty(12, dtype=torch.float32, device=cost.device)
    bc = torch.empty(1, dtype=torch.float32, device=cost.device)
    _check(lib().pilot_refine_select_best(cost.data_ptr(), poses.data_ptr(), n, idx.data_ptr(), pose.data_ptr(),
                                          bc.data_ptr(), _stream_ptr(torch, stream, cost.device)),
           "pilot_refine_select_best")
    return idx, pose, bc


def prune_topk(cost, poses, k, stream=None):
    """The k lowest-cost hypotheses in ascending (cost, index) order -> (idx int32 [k], poses [k, 12], cost [k])."""
    torch = _torch()
    n = int(cost.shape[0])
    assert cost.is_cuda and cost.dtype == torch.float32 and cost.is_contiguous() and poses.is_contiguous()
    idx = torch.empty(k, dtype=torch.int32, device=cost.device)
    po = torch.empty(k, 12, dtype=torch.float32, device=cost.device)
    co = torch.empty(k, dtype=torch.float32, device=cost.device)
    _check(lib().pilot_refine_prune_topk(cost.data_ptr(), poses.data_ptr(), n, int(k), idx.data_ptr(), po.data_ptr(),
                                         co.data_ptr(), _stream_ptr(torch, stream, cost.device)),
           "pilot_refine_prune_topk")
    return idx, po, co


# ------------------------------------------------------------------ streaming sequence

def make_frame(prob, pin=False):
    """A frame problem dict (host numpy arrays) -> (Frame struct, keep-alive list, bytes uploaded per frame).
    pin=True copies the arrays into page-locked memory once: upload() then DMAs straight from them (they must stay
    alive and unchanged until the frame was stepped)."""
    f, keep, nbytes = Frame(), [], 0
    L = int(prob["n_levels"])
    f.arrays_pinned = 1 if pin else 0
    for l in range(L):
        def hold(a, dt=None):
            a = np.ascontiguousarray(a if dt is None else np.asarray(a, dt))
            if pin and a.size:
                import torch
                t = torch.from_numpy(a.view(np.uint8).reshape(-1)).pin_memory()
                keep.append(t)
                a = t.numpy().view(a.dtype).reshape(a.shape)
            keep.append(a)
            return a
        q = hold(prob["query_feat"][l])
        f.query_feat[l] = q.ctypes.data
        nbytes += q.nbytes
        qc = prob.get("query_conf", [None] * L)[l]
        if qc is not None:
            qc = hold(qc, np.float32)
            f.query_conf[l] = qc.ctypes.data
            nbytes += qc.nbytes
        pts = hold(prob["points"][l], np.float32)
        f.n_points[l] = pts.shape[0]
        f.points[l] = pts.ctypes.data if pts.size else None
        rf = hold(prob["ref_feat"][l])
        f.ref_feat[l] = rf.ctypes.data if rf.size else None
        nbytes += pts.nbytes + rf.nbytes
        for k in range(4):
            f.intrinsics[l][k] = float(prob["intrinsics"][l][k])
    for k in range(3):
        f.gravity_imu[k] = float(prob["gravity_imu"][k])
        f.range_ray_cam[k] = float(prob["range_ray_cam"][k])
    f.range_meas = float(prob["range_meas"])
    return f, keep, nbytes


class Sequence:
    """Owns one pilot_refine_sequence: upload(frame i+1) overlaps step(frame i); everything is asynchronous until
    results() / last_frame() are read."""

    def __init__(self, n_levels, width, height, channels, dtype, n_hypotheses, max_points, total_iters, offsets,
                 dsm, dsm_origin, dsm_gsd, gravity_world, max_frames, seed_frame="camera", device=0):
        torch = _torch()
        self.torch, self.device = torch, device
        cfg = Config()
        cfg.device, cfg.n_levels, cfg.feat_dtype = device, n_levels, DTYPE_CODE[dtype]
        for l in range(n_levels):
            cfg.width[l], cfg.height[l], cfg.channels[l] = int(width[l]), int(height[l]), int(channels[l])
        cfg.max_hypotheses, cfg.max_points, cfg.max_total_iters = int(n_hypotheses), int(max_points), int(total_iters)
        sc = SequenceConfig()
        off = np.ascontiguousarray(offsets, np.float32).reshape(-1, 6)
        assert off.shape[0] == n_hypotheses
        sc.n_hypotheses, sc.offsets, sc.seed_frame = int(n_hypotheses), off.ctypes.data, SEED_CODE[seed_frame]
        if dsm is not None:
            d = np.ascontiguousarray(dsm, np.float32)
            sc.dsm, sc.dsm_height, sc.dsm_width = d.ctypes.data, d.shape[0], d.shape[1]
        sc.dsm_origin_x, sc.dsm_origin_y, sc.dsm_gsd = float(dsm_origin[0]), float(dsm_origin[1]), float(dsm_gsd)
        for k in range(3):
            sc.gravity_world[k] = float(gravity_world[k])
        sc.max_frames = int(max_frames)
        self.n_hyp, self.n_levels, self.max_frames = int(n_hypotheses), n_levels, int(max_frames)
        self.handle = C.c_void_p()
        _check(lib().pilot_refine_sequence_create(C.byref(cfg), C.byref(sc), C.byref(self.handle)),
               "pilot_refine_sequence_create")

    def _stream(self, stream):
        return _stream_ptr(self.torch, stream, self.device)

    def set_prior(self, pose, stream=None):
        p = np.ascontiguousarray(pose, np.float32).reshape(12)
        _check(lib().pilot_refine_sequence_set_prior(self.handle, p.ctypes.data, self._stream(stream)),
               "pilot_refine_sequence_set_prior")

    def upload(self, frame_prob):
        """Stage + enqueue the H2D copy of one frame (problem dict or a (Frame, keep, nbytes) tuple of make_frame)."""
        f = frame_prob if isinstance(frame_prob, tuple) else make_frame(frame_prob)
        _check(lib().pilot_refine_sequence_upload(self.handle, C.byref(f[0])), "pilot_refine_sequence_upload")
        return f[2]

    def step(self, params, stream=None):
        par, _ = make_params(params, self.n_levels)
        _check(lib().pilot_refine_sequence_step(self.handle, C.byref(par), self._stream(stream)),
               "pilot_refine_sequence_step")

    def results(self, first=0, count=None, stream=None):
        """Log rows [first, first+count) as numpy [count, 16]: pose[12], cost, best index, n_valid, status. Syncs."""
        count = self.max_frames - first if count is None else count
        out = np.zeros((count, SEQ_ROW), np.float32)
        _check(lib().pilot_refine_sequence_results(self.handle, int(first), int(count), out.ctypes.data,
                                                   self._stream(stream)), "pilot_refine_sequence_results")
        return out

    def last_frame(self, stream=None):
        """(seeds [H,12], refined poses [H,12], costs [H]) of the last stepped frame. Syncs."""
        H = self.n_hyp
        seeds, poses, cost = np.zeros((H, 12), np.float32), np.zeros((H, 12), np.float32), np.zeros(H, np.float32)
        _check(lib().pilot_refine_sequence_last_frame(self.handle, seeds.ctypes.data, poses.ctypes.data,
                                                      cost.ctypes.data, self._stream(stream)),
               "pilot_refine_sequence_last_frame")
        return seeds, poses, cost

    @property
    def last_launches(self):
        return lib().pilot_refine_sequence_last_launches(self.handle)

    def close(self):
        if self.handle:
            lib().pilot_refine_sequence_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ------------------------------------------------------------------ the paper's multi-hypothesis schedule

class PrunedRefiner:
    """supp II-C: sample H0 hypotheses around a pose prior, refine them on the coarse level, keep
    the `keep` lowest post-update objectives, refine those on the finer levels, return the arg-min.
    Five C-ABI calls per frame on one stream (seed, run_levels, prune_topk, run_levels, select_best): no host sync."""

    def __init__(self, di, params, offsets, keep, seed_frame="world", device=0):
        torch = _torch()
        self.torch, self.device, self.di, self.params = torch, device, di, dict(params)
        off = np.ascontiguousarray(offsets, np.float32).reshape(-1, 6)
        self.H0, self.keep, self.seed_frame = off.shape[0], int(keep), seed_frame
        assert 1 <= self.keep <= self.H0 <= TOPK_MAX and di.n_levels >= 2
        dev = torch.device("cuda", device)
        self.offsets = torch.from_numpy(off).to(dev)
        self.seeds = torch.empty(self.H0, 12, dtype=torch.float32, device=dev)
        P = dict(DEFAULT_PARAMS); P.update(params or {})
        self.ref = Refiner(di.n_levels, di.width, di.height, di.channels, di.dtype, self.H0, max(1, di.max_points),
                           sum(P["iters"]), device=device)
        self.inp0 = Inputs.from_buffer_copy(di.inp)
        self.inp0.n_hypotheses, self.inp0.init_poses_dev = self.H0, self.seeds.data_ptr()
        self.inp1 = Inputs.from_buffer_copy(di.inp)
        self.inp1.n_hypotheses = self.keep
        self.launches = 0

    class _View:
        def __init__(self, di, inp, n):
            self.inp, self.n_hyp, self.n_levels = inp, n, di.n_levels

    def run(self, prior_pose, stream=None, count_visible=False):
        """prior_pose: cuda float32 [12]. Returns device tensors: best_idx (into the kept set), best_pose, best_cost,
        kept_idx [keep] (into the H0 grid), poses [keep,12], cost [keep], coarse_kept_cost [keep] (ascending).
        count_visible (measurement only: synchronises twice): also `visible_evals` = [coarse level, finer levels]."""
        torch, L = self.torch, self.di.n_levels
        light = ("poses", "cost", "n_valid", "status")
        seed_hypotheses(prior_pose, self.offsets, self.seed_frame, out=self.seeds, stream=stream)
        o0 = self.ref.run(self._View(self.di, self.inp0, self.H0), self.params, stream, light, levels=(0, 1))
        n = self.ref.last_launches
        vis = [self.ref.last_visible_evals(stream)] if count_visible else None
        kept_idx, kept_poses, coarse_kept = prune_topk(o0["cost"], o0["poses"], self.keep, stream)
        self.inp1.init_poses_dev = kept_poses.data_ptr()
        o1 = self.ref.run(self._View(self.di, self.inp1, self.keep), self.params, stream, light, levels=(1, L))
        idx, pose, bc = select_best(o1["cost"], o1["poses"], stream)
        self.launches = n + self.ref.last_launches + 3
        self._keepalive = kept_poses
        if count_visible:
            vis.append(self.ref.last_visible_evals(stream))
            self.visible_evals = vis
        return dict(best_idx=idx, best_pose=pose, best_cost=bc, kept_idx=kept_idx, poses=o1["poses"], cost=o1["cost"],
                    n_valid=o1["n_valid"], status=o1["status"], coarse_kept_cost=coarse_kept)

    def close(self):
        self.ref.close()


class PrunedHostRefiner:
    """The same schedule through HOST buffers, one C call per frame (pilot_refine_submit_pruned_host / _wait_host): frame
    k+1 uploads while frame k refines. `hi` = DeviceInputs(prob, host=True) (pinned host tensors)."""

    def __init__(self, hi, params, offsets, keep, seed_frame="world", device=0):
        torch = _torch()
        self.torch, self.device, self.hi, self.keep = torch, device, hi, int(keep)
        off = np.ascontiguousarray(offsets, np.float32).reshape(-1, 6)
        self.H0, self.frame = off.shape[0], SEED_CODE[seed_frame]
        P = dict(DEFAULT_PARAMS); P.update(params or {})
        self.par, _ = make_params(params, hi.n_levels)
        dsm = (int(hi.inp.dsm_width), int(hi.inp.dsm_height))
        self.ref = Refiner(hi.n_levels, hi.width, hi.height, hi.channels, hi.dtype, self.H0, max(1, hi.max_points),
                           sum(P["iters"]), device=device, host_path=True, max_dsm=dsm)
        _check(lib().pilot_refine_set_grid_host(self.ref.handle, off.ctypes.data, self.H0), "pilot_refine_set_grid_host")
        self.res = [dict(pose=torch.zeros(12, dtype=torch.float32).pin_memory(), cost=torch.zeros(1, dtype=torch.float32).pin_memory(),
                         index=torch.zeros(1, dtype=torch.int32).pin_memory()) for _ in range(2)]
        self.priors = [torch.zeros(12, dtype=torch.float32).pin_memory() for _ in range(2)]
        self.n_sub, self.pending = 0, []

    def submit(self, prior_pose, stream=None):
        k = self.n_sub & 1
        self.priors[k].copy_(self.torch.as_tensor(np.asarray(prior_pose, np.float32).reshape(12)))
        st = stream if stream is not None else self.torch.cuda.current_stream(self.device)
        r = self.res[k]
        t = lib().pilot_refine_submit_pruned_host(self.ref.handle, C.byref(self.hi.inp), C.byref(self.par), self.priors[k].data_ptr(),
                                                  self.keep, self.frame, r["pose"].data_ptr(), r["cost"].data_ptr(),
                                                  r["index"].data_ptr(), C.c_void_p(st.cuda_stream))
        if t < 0:
            _check(t, "pilot_refine_submit_pruned_host")
        self.pending.append(k)
        self.n_sub += 1
        return t

    def wait(self):
        _check(lib().pilot_refine_wait_host(self.ref.handle), "pilot_refine_wait_host")
        return self.res[self.pending.pop(0)]

    @property
    def launches(self):
        return self.ref.last_launches

    def close(self):
        self.ref.close()


def probe_gather(buffer_bytes, vec_bytes, launches=5, device=0):
    """Random-gather bandwidth (GB/s) of the GPU for aligned vec_bytes reads from a buffer of buffer_bytes."""
    _torch()
    g = C.c_double()
    _check(lib().pilot_refine_probe_gather(int(device), int(buffer_bytes), int(vec_bytes), int(launches), C.byref(g)),
           "pilot_refine_probe_gather")
    return g.value


def probe_unit_gather(buffer_bytes, px_bytes, variant=0, launches=5, device=0):
    """Random gather of unit-shaped footprints (2 x 2 pixels of px_bytes + a reference row): GB/s of tap bytes.
    variant 0 = the kernel's LDG shape, 1 = staged through shared memory with cp.async.bulk."""
    _torch()
    g = C.c_double()
    _check(lib().pilot_refine_probe_unit_gather(int(device), int(buffer_bytes), int(px_bytes), int(variant), int(launches),
                                                C.byref(g)), "pilot_refine_probe_unit_gather")
    return g.value


# ------------------------------------------------------------------ reference-crop geometry (supp II-B)

def footprint(pose, intrinsics, width, height, dsm, dsm_origin, dsm_gsd, n_samples, s_max, stream=None):
    """supp Eq.(2). pose: cuda float32 [12]; dsm: cuda float32 [Hd, Wd]. -> cuda float32 [4, 4] (x, y, z, residual)."""
    torch = _torch()
    assert pose.is_cuda and dsm.is_cuda and pose.dtype == dsm.dtype == torch.float32 and dsm.is_contiguous()
    K = (C.c_float * 4)(*[float(k) for k in intrinsics])
    out = torch.empty(4, 4, dtype=torch.float32, device=pose.device)
    _check(lib().pilot_refine_footprint(pose.data_ptr(), K, int(width), int(height), dsm.data_ptr(), dsm.shape[1],
                                        dsm.shape[0], float(dsm_origin[0]), float(dsm_origin[1]), float(dsm_gsd),
                                        int(n_samples), float(s_max), out.data_ptr(),
                                        _stream_ptr(torch, stream, pose.device)), "pilot_refine_footprint")
    return out


def lift_anchors(corners, crop_w, crop_h, pix, dsm, dsm_origin, dsm_gsd, stream=None):
    """supp Eq.(3). corners: cuda float32 [4, 4]; pix: cuda float32 [n, 2] crop pixels -> anchors cuda float32 [n, 4]."""
    torch = _torch()
    assert corners.is_cuda and pix.is_cuda and pix.dtype == torch.float32 and pix.is_contiguous() and dsm.is_contiguous()
    n = int(pix.shape[0])
    out = torch.empty(n, 4, dtype=torch.float32, device=pix.device)
    _check(lib().pilot_refine_lift_anchors(corners.data_ptr(), int(crop_w), int(crop_h), pix.data_ptr(), n,
                                           dsm.data_ptr(), dsm.shape[1], dsm.shape[0], float(dsm_origin[0]),
                                           float(dsm_origin[1]), float(dsm_gsd), out.data_ptr(),
                                           _stream_ptr(torch, stream, pix.device)), "pilot_refine_lift_anchors")
    return out


# ------------------------------------------------------------------ unrolled reprojection supervision (supp III-C)

def reprojection_loss(poses, pose_star, points, intrinsics, width, height, z_near, alpha, scale, stream=None):
    """supp Eq.(7)-(8), forward value. poses: cuda float32 [n, 12]; pose_star: 12 host floats; points: cuda float32
    [N, 4]. -> (loss cuda float32 [n], n_visible cuda int32 [n])."""
    torch = _torch()
    assert poses.is_cuda and points.is_cuda and poses.dtype == points.dtype == torch.float32
    assert poses.is_contiguous() and points.is_contiguous()
    n = int(poses.shape[0])
    K = (C.c_float * 4)(*[float(k) for k in intrinsics])
    Ts = (C.c_float * 12)(*[float(t) for t in pose_star])
    loss = torch.empty(n, dtype=torch.float32, device=poses.device)
    nvis = torch.empty(n, dtype=torch.int32, device=poses.device)
    _check(lib().pilot_refine_reprojection_loss(poses.data_ptr(), n, Ts, points.data_ptr(), int(points.shape[0]), K,
                                                int(width), int(height), float(z_near), float(alpha), float(scale),
                                                loss.data_ptr(), nvis.data_ptr(), _stream_ptr(torch, stream, poses.device)),
           "pilot_refine_reprojection_loss")
    return loss, nvis


def reprojection_loss_grad(poses, pose_star, points, intrinsics, width, height, z_near, alpha, scale, stream=None):
    """As reprojection_loss, plus dL/d eps [n, 6] for the left perturbation of T_cw (eps = (rho; phi))."""
    torch = _torch()
    assert poses.is_cuda and points.is_cuda and poses.dtype == points.dtype == torch.float32
    n = int(poses.shape[0])
    K = (C.c_float * 4)(*[float(k) for k in intrinsics])
    Ts = (C.c_float * 12)(*[float(t) for t in pose_star])
    loss = torch.empty(n, dtype=torch.float32, device=poses.device)
    nvis = torch.empty(n, dtype=torch.int32, device=poses.device)
    grad = torch.empty(n, 6, dtype=torch.float32, device=poses.device)
    _check(lib().pilot_refine_reprojection_loss_grad(poses.data_ptr(), n, Ts, points.data_ptr(), int(points.shape[0]), K,
                                                     int(width), int(height), float(z_near), float(alpha), float(scale),
                                                     loss.data_ptr(), nvis.data_ptr(), grad.data_ptr(),
                                                     _stream_ptr(torch, stream, poses.device)), "pilot_refine_reprojection_loss_grad")
    return loss, nvis, grad


def lm_step_adjoint(hessian, gradient, lam, q, damp="identity", stream=None):
    """Adjoint of n LM steps. hessian [n, 36], gradient [n, 6], lam [n], q [n, 6] (cuda float32).
    -> dict(dxi, grad_hessian [n, 36], grad_gradient, q_prev, status)."""
    torch = _torch()
    n = int(hessian.shape[0])
    dev = hessian.device
    o = dict(dxi=torch.empty(n, 6, dtype=torch.float32, device=dev), grad_hessian=torch.empty(n, 36, dtype=torch.float32, device=dev),
             grad_gradient=torch.empty(n, 6, dtype=torch.float32, device=dev), q_prev=torch.empty(n, 6, dtype=torch.float32, device=dev),
             status=torch.empty(n, dtype=torch.int32, device=dev))
    _check(lib().pilot_refine_lm_step_adjoint(hessian.contiguous().data_ptr(), gradient.contiguous().data_ptr(),
                                              lam.contiguous().data_ptr(), q.contiguous().data_ptr(), n, DAMP_CODE[damp],
                                              o["dxi"].data_ptr(), o["grad_hessian"].data_ptr(), o["grad_gradient"].data_ptr(),
                                              o["q_prev"].data_ptr(), o["status"].data_ptr(), _stream_ptr(torch, stream, dev)),
           "pilot_refine_lm_step_adjoint")
    return o


def photo_backward(di, level, poses, grad_hessian, grad_gradient, loss="huber", loss_scale=0.1, z_near=0.1, stream=None,
                   want_conf=True):
    """Backward of the photo term of level `level` of DeviceInputs `di` (pilot_refine_photo_backward). poses [n, 12],
    grad_hessian [n, 36], grad_gradient [n, 6]: cuda float32. -> dict(grad_feat [H, W, C], grad_ref [N, C], grad_conf
    [H, W] or None, grad_pose [n, 6]) fresh, zero-initialised fp32 tensors."""
    torch = _torch()
    dev = poses.device
    Hh, W, Cn, N = di.height[level], di.width[level], di.channels[level], int(di.inp.n_points[level])
    has_conf = bool(di.inp.query_conf_dev[level]) and want_conf
    o = dict(grad_feat=torch.zeros(Hh, W, Cn, dtype=torch.float32, device=dev), grad_ref=torch.zeros(N, Cn, dtype=torch.float32, device=dev),
             grad_conf=torch.zeros(Hh, W, dtype=torch.float32, device=dev) if has_conf else None,
             grad_pose=torch.empty(int(poses.shape[0]), 6, dtype=torch.float32, device=dev))
    K = (C.c_float * 4)(*[float(di.inp.intrinsics[level][k]) for k in range(4)])
    _check(lib().pilot_refine_photo_backward(di.inp.query_feat_dev[level], di.inp.query_conf_dev[level], W, Hh, Cn, DTYPE_CODE[di.dtype],
                                             K, di.inp.points_dev[level], di.inp.ref_feat_dev[level], N, poses.contiguous().data_ptr(),
                                             grad_hessian.contiguous().data_ptr(), grad_gradient.contiguous().data_ptr(),
                                             int(poses.shape[0]), LOSS_CODE[loss], float(loss_scale), float(z_near),
                                             o["grad_feat"].data_ptr(), o["grad_ref"].data_ptr(),
                                             o["grad_conf"].data_ptr() if has_conf else None, o["grad_pose"].data_ptr(),
                                             _stream_ptr(torch, stream, dev)), "pilot_refine_photo_backward")
    return o

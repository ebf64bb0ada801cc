"""ctypes binding of the CPU oracle (oracle/pilot_oracle.c).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module. It imports nothing from the product package.
All arrays are numpy host arrays. Struct layouts mirror oracle/pilot_oracle_types.h (the oracle's own statement of the data interface).
"""
import ctypes as C
import os
import subprocess

import numpy as np

MAX_LEVELS = 4
_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = os.path.join(_HERE, "libpilot_oracle.so")

DTYPE_CODE = {"f32": 0, "bf16": 1, "f16": 2}
LOSS_CODE = {"l2": 0, "huber": 1, "cauchy": 2}
RANGE_CODE = {"off": 0, "height": 1, "march": 2}
LM_CODE = {"adaptive": 0, "fixed": 1}
DAMP_CODE = {"identity": 0, "diag": 1}
GRAD_CODE = {"bilinear_exact": 0, "central_sampled": 1}


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


class Extra(C.Structure):
    _fields_ = [("poses", C.c_void_p), ("cost", C.c_void_p), ("last_step", C.c_void_p),
                ("iter_gabs", C.c_void_p), ("iter_poses", C.c_void_p)]


def build(force=False):
    """Compile libpilot_oracle.so with gcc (building the checker is not using it)."""
    src = os.path.join(_HERE, "pilot_oracle.c")
    hdrs = [os.path.join(_HERE, "pilot_oracle.h"), os.path.join(_HERE, "pilot_oracle_types.h")]
    if not force and os.path.exists(_LIB):
        t = os.path.getmtime(_LIB)
        if all(os.path.getmtime(f) <= t for f in [src] + hdrs):
            return _LIB
    cmd = ["gcc", "-O2", "-std=c11", "-Wall", "-fPIC", "-shared", "-fopenmp", "-o", _LIB, src, "-lm"]
    subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        dp = C.POINTER(C.c_double)
        L.pilot_oracle_loss.argtypes = [C.c_int, C.c_double, C.c_double, dp, dp]
        L.pilot_oracle_loss.restype = None
        L.pilot_oracle_se3_exp.argtypes = [dp, dp, dp]
        L.pilot_oracle_se3_exp.restype = None
        L.pilot_oracle_retract.argtypes = [dp, dp, dp, dp, dp]
        L.pilot_oracle_retract.restype = None
        L.pilot_oracle_chol_solve6.argtypes = [dp, dp, dp]
        L.pilot_oracle_chol_solve6.restype = C.c_int
        L.pilot_oracle_dsm_sample.argtypes = [C.POINTER(Inputs), C.c_double, C.c_double, dp, dp, dp]
        L.pilot_oracle_dsm_sample.restype = C.c_int
        L.pilot_oracle_photo_point.argtypes = [C.POINTER(Config), C.POINTER(Inputs), C.POINTER(Params), C.c_int,
                                               dp, dp, C.c_int, dp, dp, dp, dp, dp, dp, dp]
        L.pilot_oracle_photo_point.restype = C.c_int
        L.pilot_oracle_gravity.argtypes = [C.POINTER(Inputs), dp, dp, dp]
        L.pilot_oracle_gravity.restype = None
        L.pilot_oracle_range.argtypes = [C.POINTER(Inputs), C.POINTER(Params), dp, dp, dp, dp, dp]
        L.pilot_oracle_range.restype = C.c_int
        L.pilot_oracle_eval.argtypes = [C.POINTER(Config), C.POINTER(Inputs), C.POINTER(Params), C.c_int, C.c_int,
                                        dp, dp, dp, dp, dp, C.POINTER(C.c_int), dp, C.POINTER(C.c_uint)]
        L.pilot_oracle_eval.restype = None
        L.pilot_oracle_run.argtypes = [C.POINTER(Config), C.POINTER(Inputs), C.POINTER(Params), C.POINTER(Outputs),
                                       C.POINTER(Extra), C.c_int, C.c_int, C.c_int]
        L.pilot_oracle_run.restype = C.c_int
        L.pilot_oracle_threads.argtypes = [C.c_int]
        L.pilot_oracle_threads.restype = C.c_int
        _lib = L
    return _lib


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _d(x, n=None):
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float64).reshape(-1))
    if n is not None:
        assert a.size == n, (a.size, n)
    return a


# ---------------------------------------------------------------- problem dict -> C structs
#
# A "problem" is the plain dict of numpy arrays the seeded generators
# (paper_2606_31098_b200/workloads.py) produce; see its docstring for the keys.

DEFAULT_PARAMS = dict(
    iters=[10], loss="huber", loss_scale=0.1, lm_mode="adaptive", damp_mode="identity",
    lambda_init=1e-2, lambda_up=10.0, lambda_down=0.1, lambda_min=1e-8, lambda_max=1e8,
    grad_mode="bilinear_exact", z_near=0.1, min_valid=8,
    w_gravity=0.0, gravity_scale=0.1, range_mode="off", w_range=1.0, range_scale=5.0,
    march_steps=64, bisect_steps=8, march_tfar_scale=2.0)


class Bound:
    """C structs for one problem plus the numpy arrays that keep their pointers alive."""

    def __init__(self, prob, params=None):
        self.keep = []
        L = int(prob["n_levels"])
        cfg, inp, par = Config(), Inputs(), Params()
        cfg.device = 0
        cfg.n_levels = L
        cfg.feat_dtype = DTYPE_CODE[prob["dtype"]]
        H = int(prob["init_poses"].shape[0])
        inp.n_hypotheses = H
        for l in range(L):
            cfg.width[l], cfg.height[l], cfg.channels[l] = (int(prob["width"][l]), int(prob["height"][l]),
                                                            int(prob["channels"][l]))
            q = self._hold(prob["query_feat"][l])
            assert q.size == cfg.width[l] * cfg.height[l] * cfg.channels[l]
            inp.query_feat_dev[l] = q.ctypes.data
            qc = prob.get("query_conf", [None] * L)[l]
            inp.query_conf_dev[l] = None if qc is None else self._hold(qc, np.float32).ctypes.data
            for k in range(4):
                inp.intrinsics[l][k] = float(prob["intrinsics"][l][k])
            pts = self._hold(prob["points"][l], np.float32)
            inp.n_points[l] = pts.shape[0]
            inp.points_dev[l] = pts.ctypes.data if pts.size else None
            rf = self._hold(prob["ref_feat"][l])
            assert rf.size == pts.shape[0] * cfg.channels[l]
            inp.ref_feat_dev[l] = rf.ctypes.data if rf.size else None
        poses = self._hold(prob["init_poses"], np.float32)
        inp.init_poses_dev = poses.ctypes.data if poses.size else None
        for k in range(3):
            inp.gravity_world[k] = float(prob["gravity_world"][k])
            inp.gravity_imu[k] = float(prob["gravity_imu"][k])
            inp.range_ray_cam[k] = float(prob["range_ray_cam"][k])
        inp.range_meas = float(prob["range_meas"])
        dsm = prob.get("dsm")
        if dsm is not None:
            d = self._hold(dsm, np.float32)
            inp.dsm_dev = d.ctypes.data
            inp.dsm_height, inp.dsm_width = d.shape
        inp.dsm_origin_x, inp.dsm_origin_y = float(prob["dsm_origin"][0]), float(prob["dsm_origin"][1])
        inp.dsm_gsd = float(prob["dsm_gsd"])
        P = dict(DEFAULT_PARAMS)
        P.update(prob.get("params", {}))
        if params:
            P.update(params)
        assert len(P["iters"]) == L, "params.iters needs one entry per level"
        for l in range(L):
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
        cfg.max_hypotheses, cfg.max_points = H, max(int(inp.n_points[l]) for l in range(L))
        cfg.max_total_iters = sum(int(par.iters[l]) for l in range(L))
        self.cfg, self.inp, self.par, self.P = cfg, inp, par, P
        self.H, self.L, self.total_iters = H, L, cfg.max_total_iters

    def _hold(self, a, dt=None):
        a = np.ascontiguousarray(a if dt is None else np.asarray(a, dtype=dt))
        self.keep.append(a)
        return a


def pose_to_RC(T):
    """[R_wc | C] (12,) or (3,4) -> (R_cw (9,), C (3,)) in double."""
    T = np.asarray(T, dtype=np.float64).reshape(3, 4)
    return np.ascontiguousarray(T[:, :3].T).reshape(-1), np.ascontiguousarray(T[:, 3])


def loss(kind, x, scale):
    r, d = C.c_double(), C.c_double()
    lib().pilot_oracle_loss(LOSS_CODE[kind], float(x), float(scale), C.byref(r), C.byref(d))
    return r.value, d.value


def se3_exp(xi):
    xi = _d(xi, 6)
    E, V = np.zeros(9), np.zeros(9)
    lib().pilot_oracle_se3_exp(_dptr(xi), _dptr(E), _dptr(V))
    return E.reshape(3, 3), V.reshape(3, 3)


def retract(R_cw, Cc, xi):
    R, Cv, xi = _d(R_cw, 9), _d(Cc, 3), _d(xi, 6)
    Ro, Co = np.zeros(9), np.zeros(3)
    lib().pilot_oracle_retract(_dptr(R), _dptr(Cv), _dptr(xi), _dptr(Ro), _dptr(Co))
    return Ro, Co


def chol_solve6(A, b):
    A, b = _d(A, 36), _d(b, 6)
    x = np.zeros(6)
    ok = lib().pilot_oracle_chol_solve6(_dptr(A), _dptr(b), _dptr(x))
    return bool(ok), x


def dsm_sample(bound, x, y):
    z, dx, dy = C.c_double(), C.c_double(), C.c_double()
    ok = lib().pilot_oracle_dsm_sample(C.byref(bound.inp), float(x), float(y), C.byref(z), C.byref(dx), C.byref(dy))
    return bool(ok), z.value, dx.value, dy.value


def photo_point(bound, level, R_cw, Cc, j):
    """Returns None if invisible, else dict(uv, f, gx, gy, r, Juv (2,6), w)."""
    n = int(bound.cfg.channels[level])
    R, Cv = _d(R_cw, 9), _d(Cc, 3)
    uv, f, gx, gy, r, J = np.zeros(2), np.zeros(n), np.zeros(n), np.zeros(n), np.zeros(n), np.zeros(12)
    w = C.c_double()
    ok = lib().pilot_oracle_photo_point(C.byref(bound.cfg), C.byref(bound.inp), C.byref(bound.par), level,
                                        _dptr(R), _dptr(Cv), int(j), _dptr(uv), _dptr(f), _dptr(gx), _dptr(gy),
                                        _dptr(r), _dptr(J), C.byref(w))
    if not ok:
        return None
    return dict(uv=uv, f=f, gx=gx, gy=gy, r=r, Juv=J.reshape(2, 6), w=w.value)


def gravity(bound, R_cw):
    R = _d(R_cw, 9)
    r, J = np.zeros(3), np.zeros(18)
    lib().pilot_oracle_gravity(C.byref(bound.inp), _dptr(R), _dptr(r), _dptr(J))
    return r, J.reshape(3, 6)


def range_term(bound, R_cw, Cc):
    """Returns None if skipped, else (r, J (6,), d_hit)."""
    R, Cv = _d(R_cw, 9), _d(Cc, 3)
    r, dh, J = C.c_double(), C.c_double(), np.zeros(6)
    ok = lib().pilot_oracle_range(C.byref(bound.inp), C.byref(bound.par), _dptr(R), _dptr(Cv),
                                  C.byref(r), _dptr(J), C.byref(dh))
    return (r.value, J, dh.value) if ok else None


def evaluate(bound, level, R_cw, Cc, which=7):
    R, Cv = _d(R_cw, 9), _d(Cc, 3)
    H, g = np.zeros(36), np.zeros(6)
    cost, gabs, nv, fl = C.c_double(), C.c_double(), C.c_int(), C.c_uint()
    lib().pilot_oracle_eval(C.byref(bound.cfg), C.byref(bound.inp), C.byref(bound.par), level, which,
                            _dptr(R), _dptr(Cv), _dptr(H), _dptr(g), C.byref(cost), C.byref(nv),
                            C.byref(gabs), C.byref(fl))
    return dict(H=H.reshape(6, 6), g=g, cost=cost.value, n_valid=nv.value, g_abs=gabs.value, flags=fl.value)


def run(bound, hyp_begin=0, hyp_step=1, n_threads=1):
    """Full refinement. Returns dict of numpy outputs (float32 like the C-ABI) plus double extras."""
    H, T = bound.H, bound.total_iters
    o = dict(poses=np.zeros((H, 12), np.float32), cost=np.zeros(H, np.float32),
             n_valid=np.zeros(H, np.int32), status=np.zeros(H, np.uint32),
             iter_hessian=np.zeros((T, H, 36), np.float32), iter_gradient=np.zeros((T, H, 6), np.float32),
             iter_cost=np.zeros((T, H), np.float32), iter_lambda=np.zeros((T, H), np.float32))
    e = dict(poses64=np.zeros((H, 12)), cost64=np.zeros(H), last_step=np.zeros(H),
             iter_gabs=np.zeros((T, H)), iter_poses=np.zeros((T, H, 12)))
    out, ex = Outputs(), Extra()
    out.poses_dev, out.cost_dev = o["poses"].ctypes.data, o["cost"].ctypes.data
    out.n_valid_dev, out.status_dev = o["n_valid"].ctypes.data, o["status"].ctypes.data
    out.iter_hessian_dev, out.iter_gradient_dev = o["iter_hessian"].ctypes.data, o["iter_gradient"].ctypes.data
    out.iter_cost_dev, out.iter_lambda_dev = o["iter_cost"].ctypes.data, o["iter_lambda"].ctypes.data
    ex.poses, ex.cost, ex.last_step = e["poses64"].ctypes.data, e["cost64"].ctypes.data, e["last_step"].ctypes.data
    ex.iter_gabs, ex.iter_poses = e["iter_gabs"].ctypes.data, e["iter_poses"].ctypes.data
    rc = lib().pilot_oracle_run(C.byref(bound.cfg), C.byref(bound.inp), C.byref(bound.par), C.byref(out),
                                C.byref(ex), int(hyp_begin), int(hyp_step), int(n_threads))
    if rc != 0:
        raise RuntimeError(f"pilot_oracle_run failed: {rc}")
    o.update(e)
    o["threads"] = lib().pilot_oracle_threads(int(n_threads))
    return o

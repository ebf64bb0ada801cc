"""The C-ABI library loads and exports every symbol include/pilot_refine.h declares (no compute calls)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "pilot_refine.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pilot_refine_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_2606_31098_b200 import build
    lib = ctypes.CDLL(build.build())
    names = declared_functions()
    assert {"pilot_refine_create", "pilot_refine_run", "pilot_refine_destroy"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n


def test_pure_host_entry_points():
    from paper_2606_31098_b200 import binding
    L = binding.lib()
    cfg = binding.Config()
    assert L.pilot_refine_workspace_bytes(ctypes.byref(cfg)) == 0          # bad config
    cfg.n_levels, cfg.feat_dtype = 1, 1
    cfg.width[0], cfg.height[0], cfg.channels[0] = 480, 270, 32
    cfg.max_hypotheses, cfg.max_points, cfg.max_total_iters = 64, 4096, 30
    n = L.pilot_refine_workspace_bytes(ctypes.byref(cfg))
    assert n > 64 * 16 * 128 and n % 256 == 0
    assert L.pilot_refine_destroy(None) == 0
    assert L.pilot_refine_last_launches(None) == 0
    h = ctypes.c_void_p()
    assert L.pilot_refine_create(None, ctypes.byref(h)) == -1
    assert L.pilot_refine_run(None, None, None, None, None) == -1
    # tap addresses are 32-bit byte offsets: a level map of 4 GiB or more is refused (before any CUDA call), not wrapped
    big = binding.Config()
    big.n_levels, big.feat_dtype = 1, 1
    big.width[0], big.height[0], big.channels[0] = 8192, 4096, 64           # 4 GiB of bf16
    big.max_hypotheses, big.max_points, big.max_total_iters = 4, 1024, 4
    assert L.pilot_refine_create(ctypes.byref(big), ctypes.byref(h)) == -3 and not h.value
    big.width[0] = 8191
    big.max_points = (1 << 24) + 1                                          # n_valid is summed in fp32
    assert L.pilot_refine_create(ctypes.byref(big), ctypes.byref(h)) == -3 and not h.value


def test_binding_refuses_without_gpu():
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2606_31098_b200 import binding
    from tests.small_problems import tiny
    with pytest.raises(RuntimeError):
        binding.refine(tiny())


def _data_interface(path):
    """Constants, enums and POD structs of a header as a normalised token string (comments and layout removed)."""
    src = open(path).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    items = re.findall(r"typedef\s+enum\s*\{[^}]*\}\s*\w+\s*;|typedef\s+struct\s*\{[^}]*\}\s*\w+\s*;|#define[ \t]+PILOT_\w+[ \t]+\S+", src)
    return {re.search(r"(\w+)\s*;?$|#define\s+(\w+)", it).group(0).strip(" ;"): re.sub(r"\s+", " ", it).strip() for it in items}


def test_oracle_types_describe_the_same_bytes_as_the_abi_header():
    # The oracle shares no header with the product: oracle/pilot_oracle_types.h restates the data interface. Every
    # struct, enum and constant it declares must read token for token as include/pilot_refine.h declares it.
    abi = _data_interface(os.path.join(ROOT, "include", "pilot_refine.h"))
    orc = _data_interface(os.path.join(ROOT, "oracle", "pilot_oracle_types.h"))
    for name in ("pilot_refine_config", "pilot_refine_inputs", "pilot_refine_params", "pilot_refine_outputs",
                 "pilot_dtype", "pilot_loss", "pilot_range_mode", "pilot_lm_mode", "pilot_damp_mode", "pilot_grad_mode"):
        assert name in orc and name in abi, name
    for name, text in orc.items():
        assert abi.get(name) == text, name
    assert "pilot_refine.h" not in re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "oracle", "pilot_oracle.h")).read(), flags=re.S)


def test_unrolled_backward_argument_checks_need_no_gpu():
    """pilot_refine_unrolled_backward refuses bad arguments before any CUDA call: NULL structs, priors on (their
    pose-dependence is not part of the chain), the sampled-gradient mode, missing records, a scratch buffer that is too small."""
    from paper_2606_31098_b200 import binding
    L = binding.lib()
    sb = L.pilot_refine_unrolled_backward_scratch_bytes
    assert sb(-1, 3) == 0 and sb(4, -1) == 0 and sb(0, 0) % 256 == 0
    assert 0 < sb(2, 3) <= sb(4, 3) <= sb(4, 9) and sb(4, 9) % 256 == 0
    cfg = binding.Config()
    cfg.n_levels, cfg.feat_dtype = 2, 1
    for l in range(2):
        cfg.width[l], cfg.height[l], cfg.channels[l] = 64, 48, 32
    inp = binding.Inputs()
    inp.n_hypotheses = 2
    par, _ = binding.make_params(dict(iters=[1, 2], w_gravity=0.0, range_mode="off"), 2)
    rec, sup, g = binding.UnrolledRecords(), binding.Supervision(), binding.UnrolledGrads()
    call = lambda c, i, p, r, s_, o, scratch=None, nbytes=0: L.pilot_refine_unrolled_backward(
        ctypes.byref(c) if c else None, ctypes.byref(i) if i else None, ctypes.byref(p) if p else None,
        ctypes.byref(r) if r else None, ctypes.byref(s_) if s_ else None, ctypes.byref(o) if o else None, scratch, nbytes, None)
    assert call(None, inp, par, rec, sup, g) == -1
    assert call(cfg, inp, par, None, sup, g) == -1
    assert call(cfg, inp, par, rec, sup, g) == -1                          # records and supervision points missing
    pg, _ = binding.make_params(dict(iters=[1, 2], w_gravity=1.0, range_mode="off"), 2)
    assert call(cfg, inp, pg, rec, sup, g) == -3
    pr, _ = binding.make_params(dict(iters=[1, 2], w_gravity=0.0, range_mode="march", w_range=1.0), 2)
    assert call(cfg, inp, pr, rec, sup, g) == -3
    pc, _ = binding.make_params(dict(iters=[1, 2], w_gravity=0.0, range_mode="off", grad_mode="central_sampled"), 2)
    assert call(cfg, inp, pc, rec, sup, g) == -3
    # everything present (fake non-NULL addresses, never dereferenced on this path) but no scratch: PILOT_ERR_WORKSPACE
    w = (ctypes.c_float * 3)(1 / 3, 1 / 3, 1 / 3)
    for f in ("iter_hessian_dev", "iter_gradient_dev", "iter_lambda_dev", "iter_poses_dev", "iter_accept_dev", "final_poses_dev"):
        setattr(rec, f, 256)
    sup.points_dev, sup.n_points, sup.step_weights = 256, 1, ctypes.cast(w, ctypes.POINTER(ctypes.c_float))
    assert call(cfg, inp, par, rec, sup, g) == -2
    assert call(cfg, inp, par, rec, sup, g, 256, 16) == -2
    inp.n_hypotheses = 0
    assert call(cfg, inp, par, rec, sup, g) == 0                           # nothing to do

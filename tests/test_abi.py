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

"""The C-ABI library loads on a CPU-only box and exports every symbol include/ahs.h declares (no compute calls)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_functions():
    src = open(os.path.join(ROOT, "include", "ahs.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"AHS_API\s+[\w\s\*]+?\b(ahs_\w+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = header_functions()
    for f in ("ahs_create", "ahs_step", "ahs_diagnostics", "ahs_destroy"):
        assert f in names
    assert len(names) >= 15


def test_library_exports_every_declared_symbol():
    from paper_1809_00995_b200 import binding
    lib = binding.load()
    names = header_functions()
    assert sorted(binding.SYMBOLS) == names
    for f in names:
        assert getattr(lib, f) is not None
    assert binding.load().ahs_version().decode().endswith("sm_100a")


def test_struct_layouts_match_header():
    from paper_1809_00995_b200 import binding
    # ahs_params: 4 int32 + 9 double + uint64 + ptr + size_t + ptr + 2 double ; ahs_diag: 20 x 8 bytes
    assert C.sizeof(binding.ahs_params) == 16 + 9 * 8 + 8 + 8 + 8 + 8 + 8 + 8
    assert C.sizeof(binding.ahs_diag) == 20 * 8
    assert binding.ahs_params.dx.offset == 16 and binding.ahs_params.seed.offset == 88


def test_required_bytes_and_argument_errors_need_no_gpu():
    from paper_1809_00995_b200 import binding
    assert binding.required_bytes(32, "f64") >= 15 * 32 ** 3 * 8
    assert binding.required_bytes(1024, "f32") >= 15 * 1024 ** 3 * 4
    assert binding.required_bytes(1024, "f32") < 15 * 1024 ** 3 * 4 + (1 << 24)      # 60 B/site + scratch
    assert binding.required_bytes(3, "f32") == 0
    lib = binding.load()
    assert not lib.ahs_create_ex(None)
    assert b"NULL" in lib.ahs_last_error()
    assert lib.ahs_step(None, 1) == binding.AHS_ERR_INVALID_ARG
    assert lib.ahs_destroy(None) == binding.AHS_OK
    with pytest.raises(binding.AhsError):
        binding.Simulation(32, dx=-1.0, use_torch=False)


def test_product_path_fails_loudly_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1809_00995_b200 import binding
    with pytest.raises(binding.AhsError) as e:
        binding.Simulation(32, use_torch=False)
    assert e.value.code == binding.AHS_ERR_CUDA and "no CPU fallback" in str(e.value)
    with pytest.raises(binding.AhsError):
        binding.Simulation(32, use_torch=True)


def test_package_never_imports_the_oracle():
    """The product path and the oracle share no code and neither imports the other."""
    imp = re.compile(r"^\s*(?:from|import)\s+([\w\.]+)", re.M)
    inc = re.compile(r'^\s*#\s*include\s+[<"]([^>"]+)[>"]', re.M)
    pkg = os.path.join(ROOT, "paper_1809_00995_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert not [m for m in imp.findall(txt) if m.split(".")[0] == "oracle" or "ahs_oracle" in m], fn
                assert not [m for m in inc.findall(txt) if "oracle" in m], fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", fn)).read()
            assert not [m for m in imp.findall(txt) if m.startswith("paper_1809_00995_b200")], fn
            assert not [m for m in inc.findall(txt) if "ahs" in m or "cuda" in m], fn

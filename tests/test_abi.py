"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol that
include/sst.h declares (no compute calls here)."""
import ctypes
import os
import re

from paper_2101_11489_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "sst.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sst_[a-z_]+)\s*\(", src)))


def test_library_builds_loads_and_exports_everything():
    lib_path = build.build()
    assert os.path.exists(lib_path)
    L = ctypes.CDLL(lib_path)
    names = declared_functions()
    assert {"sst_create", "sst_upload_calib", "sst_unpack_cluster", "sst_destroy"} <= set(names)
    for n in names:
        assert hasattr(L, n), f"{n} declared in sst.h but not exported"
    assert sorted(binding.EXPORTS) == names


def test_binding_struct_layout_matches_header():
    # sst_output: 4 pointers, 3 uint32 (+pad), 10 pointers, 5 pointers, uint32 (+pad), 3 pointers
    assert ctypes.sizeof(binding.sst_output) == 4 * 8 + 16 + 10 * 8 + 5 * 8 + 8 + 3 * 8
    assert ctypes.sizeof(binding.sst_config) == 28
    assert ctypes.sizeof(binding.sst_info) == 32
    assert ctypes.sizeof(binding.sst_thresholds) == 12


def test_host_side_argument_checks_need_no_gpu():
    L = binding.load()
    ctx = ctypes.c_void_p()
    cfg = binding.sst_config(0, 0, 1024, 0)          # n_feds == 0
    assert L.sst_create(ctypes.byref(cfg), ctypes.byref(ctx)) == binding.SST_ERR_INVALID_ARG
    assert L.sst_create(None, ctypes.byref(ctx)) == binding.SST_ERR_INVALID_ARG
    assert L.sst_destroy(None) == binding.SST_ERR_INVALID_ARG
    assert L.sst_status_string(binding.SST_ERR_BAD_CALIB) == b"SST_ERR_BAD_CALIB"


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2101_11489_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), fn
                assert "liboracle" not in text and "sst_oracle" not in text, fn

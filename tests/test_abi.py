"""The C-ABI library builds, loads without a GPU and exports every symbol include/vmg.h declares."""
import ctypes
import os
import re

from paper_2507_08200_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "vmg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(vmg_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported_and_bound():
    lib_path = build.build()
    lib = ctypes.CDLL(lib_path)
    decl = declared_symbols()
    assert "vmg_solve" in decl and "vmg_create" in decl and len(decl) >= 15
    for name in decl:
        assert hasattr(lib, name), f"{name} declared in include/vmg.h but not exported by libvmg.so"
    assert sorted(binding.SYMBOLS) == decl


def test_strerror_and_null_handle_paths_need_no_gpu():
    lib = binding.load()
    assert lib.vmg_strerror(0) == b"ok"
    assert b"singular" in lib.vmg_strerror(-4)
    assert lib.vmg_destroy(None) == -1
    assert lib.vmg_num_levels(None) == -1
    h = ctypes.c_void_p()
    # size validation happens before any CUDA call
    assert lib.vmg_create(ctypes.byref(h), 1, 8, 8, 1.0, 1.0, 1.0, None) == -2
    assert lib.vmg_create(ctypes.byref(h), 1030, 1030, 1030, 1.0, 1.0, 1.0, None) == -2      # 515^3 bottom
    assert lib.vmg_create(None, 8, 8, 8, 1.0, 1.0, 1.0, None) == -1


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2507_08200_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".inl")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "vmg_oracle" not in src, f

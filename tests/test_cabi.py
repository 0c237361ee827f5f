"""CPU-side checks of the boundary: the library builds for sm_100a, loads, and exports exactly
the entry points include/matgraph.h declares; the product refuses to run without a GPU (no CPU
fallback); the product never imports the oracle and vice versa."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "matgraph.h")


def _declared():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mg_[a-z_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for must in ("mg_cutoff_graph", "mg_knn_graph", "mg_update_graph", "mg_create", "mg_destroy", "mg_check"):
        assert must in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    import paper_2307_05380_b200 as m
    path = m._build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    for name in _declared():
        assert hasattr(lib, name), f"{name} declared in matgraph.h but not exported"
    assert sorted(m.EXPORTS) == _declared()
    # ... and nothing else: the dynamic symbol table holds exactly the header's mg_* functions
    nm = subprocess.run(["nm", "-D", "--defined-only", path], capture_output=True, text=True)
    if nm.returncode == 0:
        exported = sorted({line.split()[-1] for line in nm.stdout.splitlines()
                           if len(line.split()) >= 3 and line.split()[-2] in "TW" and line.split()[-1].startswith("mg_")})
        assert exported == _declared(), set(exported) ^ set(_declared())
    lib.mg_status_string.restype = ctypes.c_char_p
    assert lib.mg_status_string(0) == b"ok"
    assert b"capacity" in lib.mg_status_string(6)


def test_library_contains_sm100a_code_only():
    import paper_2307_05380_b200 as m
    out = subprocess.run(["cuobjdump", "--list-elf", m._build.build()], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    archs = set(re.findall(r"sm_\d+a?", out.stdout))
    assert archs == {"sm_100a"}, archs


def test_no_cpu_fallback():
    import torch
    import paper_2307_05380_b200 as m
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        m.Context(0)
    # straight through the C ABI as well: mg_create must fail without a device
    lib = m._lib()
    h = ctypes.c_void_p()
    assert lib.mg_create(ctypes.byref(h), 0) == 2      # MG_ERR_CUDA
    assert not h.value
    # argument errors are synchronous and do not need a device
    assert lib.mg_check(None, None) == 1               # MG_ERR_INVALID_ARG


def test_product_and_oracle_do_not_import_each_other():
    pkg = os.path.join(ROOT, "paper_2307_05380_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "mg_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2307_05380_b200" not in text.replace("paper_2307_05380_b200/csrc, include", "")
            assert "#include \"matgraph.h\"" not in text and "libmatgraph" not in text
    text = open(os.path.join(ROOT, "workloads", "crystals.py")).read()
    assert "import oracle" not in text and "paper_2307_05380_b200" not in text

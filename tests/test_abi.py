"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every function that
include/mustaforce.h declares; the binding lists exactly those; without a GPU the product fails loudly
(no CPU fallback); the product never imports the oracle."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "mustaforce.h")


def declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mf_[A-Za-z0-9_]+)\s*\(", text)))


def test_header_declares_the_contract_calls():
    names = declared_functions()
    for need in ("mf_create", "mf_set_state", "mf_step", "mf_get_state", "mf_conserved_totals"):
        assert need in names


def test_library_builds_and_exports_every_declared_symbol():
    from paper_1510_06340_b200 import build
    lib_path, strict_path = build.build()
    for path in (lib_path, strict_path):
        lib = ctypes.CDLL(path)
        for name in declared_functions():
            assert hasattr(lib, name), "%s does not export %s" % (os.path.basename(path), name)
    lib = ctypes.CDLL(lib_path)
    lib.mf_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.mf_version()


def test_binding_covers_exactly_the_header():
    from paper_1510_06340_b200 import binding
    assert sorted(binding.SIGNATURES) == declared_functions()


def test_sass_is_sm100a_only():
    from paper_1510_06340_b200 import build
    lib_path, _ = build.build()
    out = subprocess.run(["cuobjdump", "-lelf", lib_path], stdout=subprocess.PIPE, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1510_06340_b200.binding import MustaForce, MustaForceError
    with pytest.raises(MustaForceError) as ei:
        MustaForce(16, dx=0.1)
    assert "no CUDA device" in str(ei.value)


def test_product_does_not_import_the_oracle():
    code = "import sys; import paper_1510_06340_b200.binding, paper_1510_06340_b200.workloads, paper_1510_06340_b200.build; " \
           "bad=[m for m in sys.modules if m.startswith('oracle')]; assert not bad, bad"
    subprocess.run([sys.executable, "-c", code], check=True, cwd=ROOT)
    pkg = os.path.join(ROOT, "paper_1510_06340_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "mfo_" not in text and "import oracle" not in text and "from oracle" not in text, f


def test_oracle_does_not_import_the_product():
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        text = open(os.path.join(ROOT, "oracle", f), errors="ignore").read() if f.endswith((".py", ".cpp", ".h")) else ""
        assert not re.search(r"^\s*(from|import)\s+paper_1510_06340_b200", text, flags=re.M), f
        assert not re.search(r"#include\s+[\"<][^\n]*(mustaforce|mf_device|mf_types|mf_kernels)", text), f

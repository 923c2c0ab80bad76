"""CPU-side checks of the boundary: libark_m1.so builds, loads, and exports every symbol include/ark_m1.h declares.
No compute call is made here (there is no GPU on the CPU box and the library has no CPU fallback)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "ark_m1.h")).read()
    return sorted(set(re.findall(r"ARK_M1_API[^;(]*?\b(ark_m1_\w+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = _declared_symbols()
    for must in ("ark_m1_create", "ark_m1_set_state", "ark_m1_step_explicit", "ark_m1_step_implicit"):
        assert must in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2011_13926_b200 import build, binding
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    declared = _declared_symbols()
    assert len(declared) >= 15
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in ark_m1.h but not exported"
    assert sorted(binding.SYMBOLS) == declared, "binding.SYMBOLS and ark_m1.h disagree"


def test_no_oracle_import_in_the_product():
    # the product path must not route through the oracle (or any CPU fallback)
    pkg = os.path.join(ROOT, "paper_2011_13926_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "oracle_m1" not in text, f


def test_version_string_without_gpu():
    from paper_2011_13926_b200 import version
    assert "sm_100a" in version()

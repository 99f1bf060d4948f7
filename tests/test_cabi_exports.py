"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/emri.h declares (no compute calls: there is no GPU here)."""
import os
import re

from paper_2311_17174_b200 import build, emri

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols(header="emri.h"):
    txt = open(os.path.join(ROOT, "include", header)).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(emri_[a-z0-9_]+)\s*\(", txt)))


def test_library_builds_and_exports_every_declared_symbol():
    build.build()
    L = emri.load()
    names = declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), f"libemri_b200.so does not export {n}"
    assert set(names) == set(emri.EXPORTS)
    assert not [n for n in names if "probe" in n]            # measurement helpers are not part of the boundary


def test_probe_library_exports_its_header():
    """include/emri_probe.h (bench.py's peak probes) lives in a library of its own"""
    from paper_2311_17174_b200 import probe
    build.build()
    L = probe.load()
    names = declared_symbols("emri_probe.h")
    assert set(names) == set(probe.EXPORTS)
    for n in names:
        assert hasattr(L, n)


def test_strerror_and_argument_checks_need_no_gpu():
    L = emri.load()
    assert L.emri_strerror(0) == b"success"
    assert b"invalid" in L.emri_strerror(-1)
    assert b"unknown" in L.emri_strerror(-99)
    # invalid arguments are rejected before any CUDA call
    import ctypes as C
    h = C.c_void_p()
    assert L.emri_plan_create(C.byref(h), 7, 15.0, 5, 1, None) == -1      # N odd
    assert L.emri_plan_create(C.byref(h), 64, -1.0, 5, 1, None) == -1     # dt <= 0
    assert L.emri_plan_create(C.byref(h), 64, 15.0, 0, 1, None) == -1     # n_max < 1
    assert L.emri_plan_create(C.byref(h), 64, 15.0, 129, 1, None) == -1   # n_max > cap
    assert L.emri_plan_create(C.byref(h), 64, 15.0, 5, 0, None) == -1     # K_max < 1
    assert L.emri_plan_create(None, 64, 15.0, 5, 1, None) == -1
    assert L.emri_plan_destroy(None) == -1
    assert not h.value


def test_product_path_does_not_import_the_oracle():
    """the oracle is test infrastructure: nothing under the package (nor the library) references it"""
    pkg = os.path.join(ROOT, "paper_2311_17174_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "emri_o_" not in src, f

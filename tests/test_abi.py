"""CPU-only checks of the boundary: libts.so builds/loads without a GPU and exports exactly the
functions include/ts.h declares; the binding marshals what the header says; calls fail loudly
(no CPU fallback) when there is no device."""
from __future__ import annotations

import ctypes
import re
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
HEADER = ROOT / "include" / "ts.h"


def declared_functions():
    txt = re.sub(r"/\*.*?\*/", "", HEADER.read_text(), flags=re.S)
    return sorted(set(re.findall(r"\b(ts_[a-z0-9_]+)\s*\(", txt)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1208_2407_b200 import build
    return build.build()


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for n in ("ts_plan_create", "ts_evolve", "ts_norm", "ts_plan_destroy"):
        assert n in names


def test_library_exports_every_declared_symbol(libpath):
    out = subprocess.run(["nm", "-D", "--defined-only", str(libpath)], capture_output=True,
                         text=True, check=True).stdout
    exported = {ln.split()[-1] for ln in out.splitlines() if " T " in ln}
    for n in declared_functions():
        assert n in exported, n
    # nothing else of ours leaks with C linkage
    assert {e for e in exported if e.startswith("ts_")} == set(declared_functions())


def test_binding_covers_every_symbol(libpath):
    from paper_1208_2407_b200 import binding
    assert sorted(binding.SYMBOLS) == declared_functions()
    L = binding.lib()
    for n in binding.SYMBOLS:
        assert hasattr(L, n)


def test_library_contains_sm100a_code(libpath):
    out = subprocess.run(["cuobjdump", "-lelf", str(libpath)], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    assert "sm_100a" in out.stdout


def test_validation_happens_before_any_cuda_call(libpath):
    from paper_1208_2407_b200 import binding
    L = binding.lib()
    assert L.ts_plan_create(0, 4, 0, 0) is None and "nx and ny" in binding.last_error()
    assert L.ts_plan_create(4, 4, 7, 0) is None and "dtype" in binding.last_error()
    assert L.ts_plan_create(4, 4, 0, 9) is None and "boundary" in binding.last_error()
    assert L.ts_plan_create(5, 4, 0, 1) is None and "even" in binding.last_error()
    assert L.ts_evolve(None, None, None, 1.0, 0.0, 1.0, 0.0, None, 1, None) == binding.TS_EINVAL
    assert L.ts_plan_destroy(None) == binding.TS_OK


def test_no_cpu_fallback_without_a_device(libpath):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1208_2407_b200 import binding
    L = binding.lib()
    assert L.ts_plan_create(8, 8, 0, 0) is None
    assert "CUDA" in binding.last_error()
    with pytest.raises(binding.TsError):
        binding.Plan(8, 8, torch.float32, "closed")


def test_product_and_oracle_do_not_reference_each_other():
    imp = re.compile(r"^\s*(import|from)\s+(oracle|paper_1208_2407_b200)\b", re.M)
    for f in (ROOT / "paper_1208_2407_b200").rglob("*"):
        if f.suffix in (".py", ".cu", ".h", ".cuh"):
            txt = f.read_text()
            assert "ts_oracle" not in txt and "libts_oracle" not in txt, f
            assert not [m for m in imp.finditer(txt) if m.group(2) == "oracle"], f
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix in (".py", ".c", ".h"):
            txt = f.read_text()
            assert "libts.so" not in txt and "ts.h" not in txt and "#include \"ts_" not in txt, f
            assert not [m for m in imp.finditer(txt) if m.group(2) != "oracle"], f

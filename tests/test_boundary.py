"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol
include/sstep_cg.h declares; the product path fails loudly without a GPU and never touches the oracle."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "sstep_cg.h")


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sstep_cg_[a-z_]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    import paper_2501_03743_b200 as cg
    lib = cg.load_library()
    names = declared_functions()
    assert len(names) >= 16
    assert sorted(cg.EXPORTED_SYMBOLS) == names
    for name in names:
        assert hasattr(lib, name), name
    # the boundary is plain C: no C++-mangled sstep_cg symbols are exported
    out = subprocess.run(["nm", "-D", "--defined-only", cg.LIB], capture_output=True, text=True, check=True).stdout
    exported = [ln.split()[-1] for ln in out.splitlines() if " T " in ln]
    assert set(names) <= set(exported)


def test_library_contains_sm100a_code_and_bulk_copy():
    import paper_2501_03743_b200 as cg
    cg.load_library()
    cuobjdump = "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-lelf", cg.LIB], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    sass = subprocess.run([cuobjdump, "-sass", cg.LIB], capture_output=True, text=True).stdout
    assert "UBLKCP" in sass              # cp.async.bulk (TMA engine) in the staged SpMV
    assert "DFMA" in sass                # fp64 arithmetic
    assert "ACQBULK" in sass and "PREEXIT" in sass   # griddepcontrol.wait / .launch_dependents (option pdl)


def test_no_gpu_fails_loudly():
    import torch

    import paper_2501_03743_b200 as cg
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(cg.SStepCGError):
        cg.SStepCG(0)
    # and the raw C entry point reports an error instead of computing anything
    lib = cg.load_library()
    h = ctypes.c_void_p()
    assert lib.sstep_cg_create(ctypes.byref(h), 0, None) < 0 and not h.value


def test_product_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2501_03743_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower(), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2501_03743_b200 import" not in text and "import paper_2501_03743_b200" not in text
            assert "libsstepcg" not in text

"""CPU-only: the C-ABI library builds/loads and exports every symbol include/ef.h declares.
No compute calls are made."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols(name="ef.h"):
    txt = open(os.path.join(ROOT, "include", name)).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(ef_[a-z0-9_]+)\s*\(", txt)))


def dynamic_symbols(lib_path):
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", lib_path], capture_output=True, text=True, check=True).stdout
    return sorted(l.split()[-1] for l in out.splitlines() if l.split()[-1].startswith("ef_"))


def test_header_and_binding_agree():
    from paper_2410_17954_b200 import DECLARED_SYMBOLS, DIAG_SYMBOLS
    assert sorted(DECLARED_SYMBOLS) == header_symbols("ef.h")
    assert sorted(DIAG_SYMBOLS) == header_symbols("ef_diag.h")


def test_library_exports_every_declared_symbol():
    from paper_2410_17954_b200 import build as b
    b.build()
    from paper_2410_17954_b200 import exported_symbols, DECLARED_SYMBOLS
    assert sorted(exported_symbols()) == sorted(DECLARED_SYMBOLS)


def test_product_library_exports_nothing_but_the_header():
    """No bring-up backend, probe kernel or debug hook ships in libef.so: its ef_* exports are exactly include/ef.h; the
    diagnostic build adds exactly include/ef_diag.h."""
    from paper_2410_17954_b200 import build as b
    from paper_2410_17954_b200 import library_path
    b.build()
    assert dynamic_symbols(library_path()) == header_symbols("ef.h")
    b.build_diag()
    assert dynamic_symbols(library_path(diag=True)) == sorted(header_symbols("ef.h") + header_symbols("ef_diag.h"))
    import subprocess
    kernels = subprocess.run(["cuobjdump", "-elf", library_path()], capture_output=True, text=True).stdout
    assert "simt_gemm_kernel" not in kernels and "tma_fill_kernel" not in kernels


def test_product_path_does_not_touch_oracle():
    """The package never imports, reads or links anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2410_17954_b200")
    for dirpath, _, files in os.walk(pkg):
        if "build" in dirpath.split(os.sep)[-1:]:
            continue
        for fn in files:
            if fn.endswith((".py", ".cu", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), fn
                assert "moe_oracle" not in txt, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", fn)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2410_17954_b200\b", txt, flags=re.M), fn
            assert "libef" not in txt.replace("libef's", ""), fn


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("device present")
    from paper_2410_17954_b200 import MoELayerRunner
    with pytest.raises(RuntimeError):
        MoELayerRunner(1, 8, 2, 256, 512, 4)

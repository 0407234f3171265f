"""`-m "not gpu"`: the C-ABI library builds for sm_100a, loads, and exports every symbol include/fire.h declares.

No compute call is made here (there is no GPU on this box and no CPU fallback in the library)."""
import re
import subprocess

import pytest

from conftest import ROOT


@pytest.fixture(scope="module")
def lib_path():
    from paper_1701_03549_b200 import build
    return build.build()


def declared_symbols():
    text = (ROOT / "include" / "fire.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fire_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for name in ("fire_landscape_create", "fire_params_upload", "fire_simulate_batch", "fire_fitness"):
        assert name in syms


def test_library_exports_every_declared_symbol(lib_path):
    out = subprocess.run(["nm", "-D", "--defined-only", str(lib_path)], capture_output=True, text=True, check=True).stdout
    exported = {line.split()[-1] for line in out.splitlines() if " T " in line}
    missing = [s for s in declared_symbols() if s not in exported]
    assert not missing, f"declared in fire.h but not exported: {missing}"


def test_binding_covers_the_header_and_loads(lib_path):
    from paper_1701_03549_b200 import libfire as lf
    assert sorted(lf.SYMBOLS) == declared_symbols()
    lib = lf.load()
    for s in lf.SYMBOLS:
        assert hasattr(lib, s) and callable(getattr(lf, s if s != "fire_error_string" else "error_string"))
    assert lf.error_string(lf.FIRE_OK) == "ok" and "invalid" in lf.error_string(lf.FIRE_EINVAL)


def test_header_is_valid_c99_and_prototypes_match(tmp_path):
    """include/fire.h through a C compiler (not a regex): tests/c/abi_c99.c includes it, assigns every declared call to a
    function pointer of the documented prototype and names every error / metric code."""
    src = ROOT / "tests" / "c" / "abi_c99.c"
    res = subprocess.run(["gcc", "-std=c99", "-pedantic", "-Wall", "-Wextra", "-Werror", "-I", str(ROOT / "include"),
                          "-c", str(src), "-o", str(tmp_path / "abi_c99.o")], capture_output=True, text=True)
    assert res.returncode == 0, res.stderr
    text = src.read_text()
    for name in declared_symbols():
        assert re.search(rf"=\s*{name}\s*;", text), f"{name} is not referenced by tests/c/abi_c99.c"


def test_library_is_built_for_sm_100a(lib_path):
    out = subprocess.run(["cuobjdump", "-lelf", str(lib_path)], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_product_does_not_reference_the_oracle():
    """The CUDA path and its binding never import, link or call anything under oracle/, and vice versa."""
    pkg = ROOT / "paper_1701_03549_b200"
    for f in pkg.rglob("*.py"):
        txt = f.read_text()
        assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
        assert "libfire_oracle" not in txt and "fire_oracle" not in txt, f
    for f in [*pkg.rglob("*.cu"), *pkg.rglob("*.cuh"), ROOT / "include" / "fire.h"]:
        txt = f.read_text()
        assert not re.search(r"#include\s*[<\"][^>\"]*oracle", txt) and "orc_" not in txt, f
    for f in (ROOT / "oracle").iterdir():
        if f.suffix in (".c", ".py", ".h"):
            txt = f.read_text()
            assert "libfire_sm100a" not in txt and "import libfire" not in txt and '#include "fire' not in txt, f


def test_no_gpu_means_error_not_fallback(lib_path):
    import torch
    if torch.cuda.is_available():
        pytest.skip("this box has a GPU")
    from paper_1701_03549_b200 import libfire as lf
    with pytest.raises((lf.FireError, TypeError)):
        lf.fire_landscape_create(torch.zeros((4, 4), dtype=torch.uint8), torch.zeros((4, 4)), torch.zeros((4, 4)),
                                 torch.zeros((4, 4)))

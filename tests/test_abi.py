"""The C-ABI library builds, loads, and exports every symbol include/scape.h declares (CPU only:
no compute call is made here)."""
import ctypes
import os
import re
import shutil

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "scape.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(scape_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2607_01678_b200 import build
    if build.needs_build():
        if not (os.path.exists("/usr/local/cuda/bin/nvcc") or shutil.which("nvcc")):
            pytest.skip("libscape.so not built and nvcc unavailable")
        build.build()
    return build.LIB


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for must in ("scape_create", "scape_step", "scape_destroy"):
        assert must in syms


def test_library_exports_every_declared_symbol(libpath):
    L = ctypes.CDLL(libpath)
    for name in declared_symbols():
        assert hasattr(L, name), f"{name} declared in include/scape.h but not exported"


def test_binding_covers_every_declared_symbol(libpath):
    from paper_2607_01678_b200 import binding
    assert sorted(binding.SYMBOLS) == declared_symbols()
    for name in declared_symbols():
        if name not in ("scape_last_error",):
            assert hasattr(binding, name), f"binding lacks {name}"


def test_invalid_arguments_are_rejected_without_a_gpu(libpath):
    """Argument validation happens before any CUDA call, so it is testable here."""
    from paper_2607_01678_b200 import binding
    L = binding.lib()
    assert not L.scape_create(0, 1, 0.5, 0.9, 0.95, 1e-8, 1e-3, 0.1)
    assert not L.scape_create(16, 1, 1.0, 0.9, 0.95, 1e-8, 1e-3, 0.1)
    assert not L.scape_create(16, 99, 0.5, 0.9, 0.95, 1e-8, 1e-3, 0.1)
    assert binding.scape_last_error() != ""
    assert L.scape_step(None, None, None, None) == binding.SCAPE_EINVAL
    L.scape_destroy(None)


def test_no_cpu_fallback_without_a_device(libpath):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2607_01678_b200 import binding
    with pytest.raises(binding.ScapeError):
        binding.scape_create(1024, 2, 0.9, 0.9, 0.95, 1e-8, 1e-3, 0.1)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_01678_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "liboracle" not in text, f

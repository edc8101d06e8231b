"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol include/hydro.h
declares; the binding declares the same set.  No compute calls (there is no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "hydro.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hydro_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1511_02137_b200 import build
    return build.build()


def test_header_symbols_exported(libpath):
    names = _declared_symbols()
    assert "hydro_create" in names and "hydro_step" in names and len(names) >= 15
    lib = ctypes.CDLL(libpath)
    for n in names:
        assert hasattr(lib, n), "libhydro.so does not export " + n


def test_binding_declares_the_same_symbols(libpath):
    from paper_1511_02137_b200 import hydro
    assert sorted(hydro.SYMBOLS) == _declared_symbols()
    L = hydro.load()
    assert L.hydro_strerror(0) == b"ok" and L.hydro_strerror(1) == b"invalid argument"


def test_argument_validation_without_gpu(libpath):
    """EINVAL paths return before any CUDA call."""
    from paper_1511_02137_b200 import hydro
    L = hydro.load()
    h = ctypes.c_void_p()
    assert L.hydro_create(ctypes.byref(h), 0, 8, 8, 0.1, 0.02, None, None) == hydro.EINVAL
    assert L.hydro_create(ctypes.byref(h), 8, 8, 8, -0.1, 0.02, None, None) == hydro.EINVAL
    eos = hydro.EosT(0, 3, 64, 0, 0, 0)
    assert L.hydro_create(ctypes.byref(h), 8, 8, 8, 0.1, 0.02, ctypes.byref(eos), None) == hydro.EINVAL
    eos = hydro.EosT(0, 4, 16, 0, 0, 0)
    assert L.hydro_create(ctypes.byref(h), 8, 8, 8, 0.1, 0.02, ctypes.byref(eos), None) == hydro.EINVAL
    assert L.hydro_step(None, 1) == hydro.EINVAL
    assert L.hydro_set_state(None, None, 0) == hydro.EINVAL
    assert L.hydro_launch_count(None) == -1


def test_no_cpu_fallback_without_device(libpath):
    """Without a CUDA device the product path must fail loudly, never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1511_02137_b200 import hydro
    with pytest.raises(hydro.HydroError) as e:
        hydro.Hydro(8, 8, 8, 0.1, 0.02)
    assert e.value.code == hydro.ECUDA


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1511_02137_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f

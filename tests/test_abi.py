"""CPU-side checks of the boundary (-m "not gpu"): the C-ABI library builds, loads and exports
every symbol include/tt.h declares; no compute call is made without a GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2606_06511_b200 import build
    return build.build()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "tt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tt_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for n in ("tt_energy", "tt_energy_grad_hess", "tt_hess_vec", "tt_hess_symbolic", "tt_create", "tt_destroy"):
        assert n in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(str(lib_path))
    for name in declared_functions():
        assert hasattr(lib, name), "libtt.so does not export %s" % name


def test_binding_covers_the_header(lib_path):
    from paper_2606_06511_b200 import tt
    assert sorted(tt.EXPORTS) == declared_functions()
    lib = tt.load_library()
    assert lib.tt_status_string(0) == b"TT_OK"
    assert lib.tt_status_string(-4) == b"TT_ERR_CAPACITY"


def test_no_cpu_fallback(lib_path):
    import torch
    from paper_2606_06511_b200 import tt
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        tt.Context()


def test_product_does_not_import_oracle():
    """The CUDA path and its binding never import, link or read anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_2606_06511_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "tt_oracle" not in txt, f

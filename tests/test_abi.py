"""CPU-side checks of the boundary: libdsmc.so builds, loads without a GPU and exports every symbol
include/dsmc.h declares; host-only calls behave; the oracle and the CUDA path share nothing."""
import os
import re
import ctypes

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1211_6234_b200 import build, dsmc
    build.build()
    return dsmc.load_library()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "dsmc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dsmc_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported_and_bound(lib):
    from paper_1211_6234_b200 import dsmc
    names = declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(n for n, _, _ in dsmc.ABI) == names          # the binding covers the whole header


def test_host_only_calls(lib):
    assert lib.dsmc_version().startswith(b"dsmc")
    assert lib.dsmc_workspace_bytes(7, 1) == 0                   # odd L
    assert lib.dsmc_workspace_bytes(2, 1) == 0                   # L < 4
    assert lib.dsmc_workspace_bytes(8, 0) == 0
    b1, b2 = lib.dsmc_workspace_bytes(8, 1), lib.dsmc_workspace_bytes(256, 64)
    assert 0 < b1 < b2 < 2 * 1024 ** 3
    h = ctypes.c_void_p()
    assert lib.dsmc_create(ctypes.byref(h), 7, 1, 1.0, 0.1, 0.5, 0.0) == -1 and not h
    assert lib.dsmc_create(ctypes.byref(h), 8, 2, 1.0, 0.1, 0.5, 0.0) == 0 and h
    # unbound context: every device call refuses with DSMC_ESTATE, nothing crashes
    assert lib.dsmc_build_tensor(h, 1, 0, 0) == -2
    assert lib.dsmc_halfsweep(h, None, 1, 0) == -2
    assert b"not bound" in lib.dsmc_last_error(h)
    assert lib.dsmc_select_field_kernel(h, 5) == -1
    assert lib.dsmc_launch_count(h) == 0
    assert lib.dsmc_destroy(h) == 0


def test_product_has_no_oracle_dependency():
    """The product path must not import, link or call anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1211_6234_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower(), (f, "mentions the oracle")
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1211_6234_b200" not in text and "libdsmc" not in text
            assert "#include \"../paper" not in text


def test_no_gpu_means_loud_failure():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1211_6234_b200 import Dsmc, DsmcError
    with pytest.raises(DsmcError):
        Dsmc(8, 1)

"""The C-ABI library loads and exports every symbol include/ssp.h declares (no GPU needed)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2604_07248_b200 import build, api
    build.build()
    return api.load()


def _declared():
    src = open(os.path.join(ROOT, "include", "ssp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ssp_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    from paper_2604_07248_b200 import api
    names = _declared()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), f"{n} declared in ssp.h but not exported"
    assert sorted(api.SYMBOLS) == names          # the binding knows every entry point, and no others


def test_version_and_workspace_without_gpu(lib):
    from paper_2604_07248_b200 import api
    assert "sm_100a" in api.version()
    small = api.workspace_bytes(128, 1e-3, 4, 5)
    big = api.workspace_bytes(1024, 1e-3, 32, 20)
    assert 0 < small < big
    assert big >= 64 * 1024 * 1024 * 8                    # holds a chunk of column-transformed screens
    assert api.workspace_bytes(100, 1e-3, 1, 1) == 0      # N not a power of two
    assert api.workspace_bytes(8192, 1e-3, 1, 1) == 0


def test_create_fails_loudly_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = C.c_void_p()
    rc = lib.ssp_create(C.byref(h), 0, None)
    assert rc < 0 and not h.value
    from paper_2604_07248_b200 import api
    with pytest.raises(RuntimeError):
        api.Context(0)


def test_no_oracle_in_product():
    """The product path never imports, links or calls the oracle."""
    pkg = os.path.join(ROOT, "paper_2604_07248_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("CPU oracle", "").replace("the oracle", "") or f == "synth.py", f
                assert "orc_" not in txt, f

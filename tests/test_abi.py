"""Host-side checks that need no GPU: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/ch.h declares; host-only calls (ch_init argument checks, ch_workspace_bytes,
ch_padded_cells) behave as the header says; the product refuses to run without a CUDA device."""
import ctypes
import os
import re

import pytest

import paper_1410_4194_b200 as pkg
from paper_1410_4194_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    binding.build()
    return binding.load_library()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "ch.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ch_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_symbols()
    assert set(names) == set(binding.SYMBOLS)
    for n in names:
        assert getattr(lib, n) is not None


def test_sass_is_sm_100a():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", binding._LIB], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_host_only_calls(lib):
    assert not lib.ch_init(0, 1, 1, 3, 1.4, None)
    assert not lib.ch_init(8, 8, 8, 2, 1.4, None)
    assert not lib.ch_init(8, 8, 8, 3, 0.9, None)
    assert not lib.ch_init(8, 2, 8, 3, 1.4, None)          # active dimension thinner than the ghost depth
    bc = (ctypes.c_int * 6)(1, 3, 1, 1, 1, 1)
    assert not lib.ch_init(8, 8, 8, 3, 1.4, bc)
    assert b"periodic" in lib.ch_last_error()
    bc = (ctypes.c_int * 6)(7, 7, 1, 1, 1, 1)
    assert not lib.ch_init(8, 8, 8, 3, 1.4, bc)
    h = lib.ch_init(10, 6, 1, 3, 1.4, None)
    assert h
    assert lib.ch_padded_cells(h) == 16 * 12 * 1
    assert lib.ch_workspace_bytes(10, 6, 1, 3) >= 16 * 12 * 5 * 8
    assert lib.ch_workspace_bytes(10, 6, 1, 2) == 0
    assert lib.ch_set_spacing(h, 0.0, 1.0, 1.0) == binding.CH_EINVAL
    assert lib.ch_set_spacing(h, 0.1, 0.1, 0.1) == binding.CH_OK
    assert lib.ch_step(h, 0.1) == binding.CH_ESTATE
    assert lib.ch_free(h) == binding.CH_OK


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        pkg.Grid(8, 8, 8)


def test_product_does_not_import_the_oracle():
    for root, _, files in os.walk(os.path.join(ROOT, "paper_1410_4194_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(root, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "cholla_ref" not in src, f


def test_sass_holds_the_tma_pipeline():
    """The fused second half streams its planes with TMA: the built library must contain bulk tensor loads
    (UTMALDG.4D, the SASS of cp.async.bulk.tensor.4d) and mbarrier phase checks (SYNCS...TRYWAIT)."""
    import subprocess
    out = subprocess.run(["cuobjdump", "-sass", binding._LIB], capture_output=True, text=True).stdout
    assert "UTMALDG.4D" in out and "SYNCS.PHASECHK.TRANS64.TRYWAIT" in out
    assert "MUFU.RSQ64H" in out and "MUFU.RCP64H" in out          # the branch-free rsqrt / rcp seeds

"""C-ABI checks that need no GPU: the library builds, loads and exports every symbol
include/dfjk.h declares; argument validation and the no-device failure are loud."""
import ctypes
import re

import numpy as np
import pytest

import paper_2506_06661_b200 as pkg


@pytest.fixture(scope="module")
def L():
    pkg.build()
    return pkg.lib()


def test_header_symbols_match_exports(L):
    src = open(pkg.HEADER_PATH).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    declared = set(re.findall(r"\b(dfjk_[a-z_]+)\s*\(", src))
    assert declared == set(pkg.SYMBOLS)
    for name in declared:
        assert hasattr(L, name), name
    raw = ctypes.CDLL(pkg.LIB_PATH)
    for name in declared:
        getattr(raw, name)


def test_version_and_null_handling(L):
    assert re.fullmatch(rb"\d+\.\d+\.\d+", L.dfjk_version())
    assert L.dfjk_destroy(None) == 0
    assert L.dfjk_workspace_bytes(None) == 0
    assert L.dfjk_get_jk(None, None, 1, None, None, None) == -1
    assert b"NULL handle" in L.dfjk_last_error()
    assert L.dfjk_get_jk_host(None, None, 1, None, None) == -1
    assert L.dfjk_get_jk_u_host(None, None, 1, None, 1, None, None, None) == -1
    assert L.dfjk_set_option(None, b"k_chunk", 1) == -1
    # general-density entry points (section 8f rank 1)
    assert L.dfjk_get_jk_pair(None, None, None, 1, None, None, None) == -1
    assert b"NULL" in L.dfjk_last_error()
    assert L.dfjk_get_jk_dm(None, None, None, None, None) == -1
    assert L.dfjk_get_jk_dms(None, 1, None, None, None, None) == -1
    assert L.dfjk_get_jk_pairs(None, 1, None, None, None, None, None, None) == -1
    assert b"NULL handle" in L.dfjk_last_error()
    assert L.dfjk_get_df_diag(None, None, None) == -1
    # the allocation-free entry point: argument checks come before any CUDA call
    assert L.dfjk_noalloc_max_nao() == 1023
    assert L.dfjk_df_diag_noalloc(4, 4, None, None, None) == -1
    assert b"NULL" in L.dfjk_last_error()
    assert L.dfjk_df_diag_noalloc(0, 4, None, None, None) == -1
    assert L.dfjk_df_diag_noalloc(4, 1024, None, None, None) == -1
    assert b"1023" in L.dfjk_last_error() and b"scratch" in L.dfjk_last_error()
    assert L.dfjk_scf_rhf(None, None, None, 1, 1, 1e-8, 4, None, None, None, None, None, None, None, None) == -1
    assert b"NULL handle" in L.dfjk_last_error()
    assert L.dfjk_probe_dmma_peak(None) == -1
    assert L.dfjk_build_b(0, 4, None, None, None, None) == -1
    assert L.dfjk_build_b(4, 4, None, None, None, None) == -1
    assert b"NULL" in L.dfjk_last_error()


def test_create_rejects_bad_arguments_without_touching_memory(L):
    buf = np.zeros(64)
    assert not L.dfjk_create(0, 4, buf.ctypes.data)
    assert b"naux" in L.dfjk_last_error()
    assert not L.dfjk_create(4, 0, buf.ctypes.data)
    assert not L.dfjk_create(4, 4, None)
    assert b"NULL" in L.dfjk_last_error()
    assert not L.dfjk_create(4, 4, buf.ctypes.data | 8)
    assert b"aligned" in L.dfjk_last_error()


def test_no_cpu_fallback():
    """A host pointer (or a box without a GPU) must fail loudly, never compute on the CPU."""
    L = pkg.lib()
    buf = np.zeros(4 * 10 + 2)
    ptr = (buf.ctypes.data + 15) & ~15
    assert not L.dfjk_create(4, 4, ptr)
    msg = L.dfjk_last_error()
    assert b"device" in msg.lower()
    import torch
    with pytest.raises(ValueError):
        pkg.DFJK(torch.zeros(4, 10, dtype=torch.float64), 4)


def test_product_does_not_import_oracle():
    import os
    root = os.path.dirname(pkg.__file__)
    for dirpath, _, files in os.walk(root):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp", ".c")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text
                assert "dfjk_oracle" not in text and "liboracle" not in text

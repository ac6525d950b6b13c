"""CPU-side checks of the boundary: libbh.so builds for sm_100a, loads without a GPU and exports
every symbol include/bh.h declares; compute calls fail loudly (no CPU fallback) when no device exists."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "bh.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bh_[a-z_]+)\s*\(", src)))


def test_header_and_binding_agree():
    import paper_1509_07370_b200 as pkg
    assert sorted(pkg.EXPORTED_SYMBOLS) == _declared_symbols()


def test_library_exports_every_declared_symbol():
    import paper_1509_07370_b200 as pkg
    L = pkg.lib()
    assert os.path.exists(pkg.lib_path())
    for name in _declared_symbols():
        assert hasattr(L, name), name


def test_strerror_and_stats_layout():
    import paper_1509_07370_b200 as pkg
    L = pkg.lib()
    assert L.bh_strerror(0) == b"ok"
    assert b"invalid" in L.bh_strerror(-1)
    # struct bh_stats: 3*8 + 2*4 + 6*8 + 8 + 7*4 + 3*4 + 8 bytes; struct bh_pass: 24 + 4 (+4 pad) + 8
    assert C.sizeof(pkg.Stats) == 136
    from paper_1509_07370_b200.binding import Pass
    assert C.sizeof(Pass) == 40


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    import paper_1509_07370_b200 as pkg
    L = pkg.lib()
    h = C.c_void_p()
    assert L.bh_create(C.byref(h), 0, None) == -3      # BH_ERR_CUDA
    assert not h
    with pytest.raises(Exception):
        pkg.Context(0)


def test_null_arguments_are_rejected():
    import paper_1509_07370_b200 as pkg
    L = pkg.lib()
    assert L.bh_create(None, 0, None) == -1
    assert L.bh_build(None, None, None, None, None, 10, None) == -1
    assert L.bh_potential(None, 0.5, 1.0, None) == -1
    assert L.bh_get_stats(None, None) == -1
    assert L.bh_destroy(None) == 0

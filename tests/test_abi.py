"""The C-ABI library: builds for sm_100a, loads, exports every symbol include/sup.h declares, validates arguments on
the host, and FAILS LOUDLY without a CUDA device (no CPU fallback).  No compute call is made here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "sup.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sup_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for need in ["sup_create", "sup_project_simultaneous", "sup_block_iterative", "sup_perturb_tv", "sup_perturb_dose",
                 "sup_superiorize", "sup_proximity", "sup_objective"]:
        assert need in names


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2606_27086_b200.build import build_lib

    path = build_lib()
    L = ctypes.CDLL(path)
    for name in declared_symbols():
        assert hasattr(L, name), f"{name} declared in include/sup.h but not exported by libsup.so"
    L.sup_version.restype = ctypes.c_char_p
    assert b"sm_100a" in L.sup_version()


def test_sass_is_sm100a():
    from paper_2606_27086_b200.build import LIB, build_lib

    build_lib()
    import subprocess

    out = subprocess.run(["cuobjdump", "-lelf", LIB], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_workspace_query_and_host_side_argument_checks():
    import paper_2606_27086_b200 as sup

    p, s = sup.sup_workspace_bytes(0, 1000, 500, 20000, sup.F32)
    assert p % 256 == 0 and s % 256 == 0 and p > 20000 * 8 and s > 20000 * 8
    p64, _ = sup.sup_workspace_bytes(0, 1000, 500, 20000, sup.F64)
    # fp32 handles hold A^T (8 B/nnz) plus the packed copies of A and A^T (16 B/nnz); fp64 handles A^T (12 B/nnz) + colg
    assert p >= 20000 * 24 and p64 >= 20000 * 16
    with pytest.raises(sup.SupError) as e:
        sup.sup_workspace_bytes(0, 0, 500, 10)
    assert e.value.status == 1
    with pytest.raises(sup.SupError):
        sup.sup_workspace_bytes(7, 10, 10, 10)


def test_no_cpu_fallback_without_a_device():
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import numpy as np

    import paper_2606_27086_b200 as sup
    from paper_2606_27086_b200.binding import _Csr, lib

    with pytest.raises(sup.SupError) as e:  # the binding refuses before any marshalling
        sup.sup_create(np.array([0, 1]), np.array([0], np.int32), np.ones(1, np.float32), np.zeros(1), np.ones(1), np.zeros(1), np.ones(1))
    assert e.value.status == 4
    # and so does the C entry point itself (fake, never dereferenced, 256-aligned device addresses)
    L = lib()
    A = _Csr(4, 4, 4, 0x10000, 0x20000, 0x30000)
    h = ctypes.c_void_p(None)
    rc = L.sup_create(ctypes.byref(h), ctypes.byref(A), 0x40000, 0x50000, 0x60000, 0x70000, None, 0, 0x100000, 1 << 30, 0x80000000, 1 << 30, None)
    assert rc == 4 and not h.value
    assert b"no usable CUDA device" in L.sup_last_error(None)

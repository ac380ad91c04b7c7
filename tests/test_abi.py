"""`-m "not gpu"` checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every symbol that
include/agate.h declares, sizes its workspace correctly, validates arguments, and fails loudly (AGATE_ERR_CUDA)
instead of falling back when there is no CUDA device.  No compute calls are made here."""
import ctypes as C
import os
import re

import pytest

import paper_2503_20899_b200 as ag

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "agate.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(agate_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    L = ag.lib()
    names = declared_symbols()
    assert len(names) >= 15
    for n in names:
        assert hasattr(L, n), f"libagate.so does not export {n}"
    assert sorted(ag.SYMBOLS) == names


def test_workspace_bytes_and_argument_checks():
    L = ag.lib()
    g = ag.Grid(3, 512, 512, 512, 1 / 512, 1 / 512, 1 / 512)
    s = ag.SolverCfg(ag.HLLD, 2, 1.3, 2, 0.0, 0.0)
    n = L.agate_workspace_bytes(C.byref(g), ag.IDEAL, C.byref(s))
    padded = 8 * 8 * 516 ** 3
    assert 2 * padded <= n <= 2 * padded + (1 << 20)          # two ghost-padded copies of U + scalars
    bad = ag.SolverCfg(ag.HLLD, 2, 1.3, 2, 0.0, 0.05)
    assert L.agate_workspace_bytes(C.byref(g), ag.HALL, C.byref(bad)) == 0     # Hall + HLLD is rejected
    g2 = ag.Grid(2, 64, 64, 2, 1.0, 1.0, 1.0)
    assert L.agate_workspace_bytes(C.byref(g2), ag.IDEAL, C.byref(s)) == 0     # inactive dimension must be 1
    s3 = ag.SolverCfg(ag.HLL, 2, 2.5, 2, 0.0, 0.0)
    assert L.agate_workspace_bytes(C.byref(g), ag.IDEAL, C.byref(s3)) == 0     # beta outside [1,2]
    assert L.agate_strerror(ag.ERR_UNPHYSICAL).decode().startswith("unphysical")


def test_no_cpu_fallback_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    L = ag.lib()
    g = ag.Grid(2, 32, 32, 1, 1 / 32, 1 / 32, 1.0)
    s = ag.SolverCfg(ag.HLL, 2, 1.0, 2, 0.4, 0.0)
    n = L.agate_workspace_bytes(C.byref(g), ag.IDEAL, C.byref(s))
    buf = (C.c_char * (n + 256))()
    addr = (C.addressof(buf) + 255) & ~255
    h = C.c_void_p()
    rc = L.agate_init(C.byref(g), 5 / 3, ag.IDEAL, C.byref(s), C.c_void_p(addr), n, None, C.byref(h))
    assert rc == ag.ERR_CUDA
    with pytest.raises(RuntimeError):
        ag.Agate(shape=(32, 32, 1), dx=(1 / 32, 1 / 32, 1.0), ndim=2)
    v = C.c_double()
    assert L.agate_measure_fp64_peak(1, C.byref(v), C.c_void_p(addr), None) == ag.ERR_CUDA
    assert L.agate_measure_fp64_peak(1, C.byref(v), None, None) == ag.ERR_ARG        # the caller supplies the scratch

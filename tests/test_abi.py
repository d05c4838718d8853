"""The C-ABI library builds for sm_100a, loads, and exports every symbol include/dmrg_b200.h declares (no compute)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols(header="dmrg_b200.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dmrg_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib):
    names = declared_symbols()
    assert len(names) >= 15
    dll = ctypes.CDLL(lib.binding.LIB_PATH)
    for n in names:
        assert hasattr(dll, n), "missing export " + n
    assert sorted(lib.binding.EXPORTS) == names
    # the measurement-only companion library: its own header, its own .so; the product library carries none of it
    bench = ctypes.CDLL(os.path.join(os.path.dirname(lib.binding.LIB_PATH), "libdmrg_b200_bench.so"))
    for n in declared_symbols("dmrg_b200_bench.h"):
        assert hasattr(bench, n), "missing export " + n
        assert not hasattr(dll, n)


def test_default_options_and_argument_errors_need_no_gpu(lib):
    o = lib.dmrg_default_options()
    assert o.davidson_tol == 1e-7 and o.davidson_max_subspace == 20 and o.keep_env_stack == 1
    import numpy as np
    h = np.zeros((2, 2))
    eri = np.zeros((2, 2, 2, 2))
    ctx = ctypes.c_void_p()
    f = lib.binding.lib.dmrg_create
    bad = [(0, 0, 0), (2, 5, 1), (2, 3, 0), (2, 2, 4)]            # k<1, n_elec>2k, odd n+2Sz, |2Sz| too large
    for (k, n, s2) in bad:
        rc = f(ctypes.byref(ctx), k, n, s2, h.ctypes.data_as(ctypes.c_void_p), eri.ctypes.data_as(ctypes.c_void_p), None)
        assert rc == lib.DMRG_EINVAL
    h[0, 1] = 1.0                                                  # asymmetric h
    rc = f(ctypes.byref(ctx), 2, 2, 0, h.ctypes.data_as(ctypes.c_void_p), eri.ctypes.data_as(ctypes.c_void_p), None)
    assert rc == lib.DMRG_EINVAL

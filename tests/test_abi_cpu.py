"""CPU-side checks of the C-ABI library: it builds, loads, exports every symbol include/clt.h declares, its host
logic validates arguments, and it fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1812_00525_b200 import build as clt_build
from paper_1812_00525_b200 import clt

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    clt_build.build()
    return clt.load()


def test_header_symbols_are_all_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "clt.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = sorted(set(re.findall(r"\b(clt_[A-Za-z_0-9]+)\s*\(", hdr)))
    assert len(names) >= 21
    assert sorted(clt.EXPORTS) == names
    for n in names:
        assert hasattr(lib, n), n


def test_strerror_and_version(lib):
    assert lib.clt_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4, -5):
        assert len(lib.clt_strerror(code)) > 3
    assert b"sm_100a" in lib.clt_version()


def test_workspace_bytes_and_grid_validation(lib):
    g = clt.clt_grid(512, 64, 512, 2.0, 4.0, -1.0, 1.0, 0.0)
    nbytes = lib.clt_workspace_bytes(ctypes.byref(g))
    dense38 = 38 * 512 * 64 * 512 * 8
    # 35 fields + 3 for the Hall field G (NEXT-3) + padding + small tables
    assert dense38 <= nbytes <= 1.06 * dense38
    for bad in (clt.clt_grid(8, 64, 512, 2, 4, -1, 1, 0), clt.clt_grid(512, 4, 512, 2, 4, -1, 1, 0),
                clt.clt_grid(512, 64, 512, 0.0, 4, -1, 1, 0), clt.clt_grid(512, 64, 512, 2, 4, 1, -1, 0),
                clt.clt_grid(512, 64, 512, 2, 1, -1, 1, 0)):
        assert lib.clt_workspace_bytes(ctypes.byref(bad)) == 0


def test_null_and_bad_arguments_are_rejected(lib):
    g = clt.clt_grid(32, 16, 32, 2.0, 4.0, -1.0, 1.0, 0.0)
    p = clt.clt_params(5 / 3, 1e-5, 1e-5, 1e-5, 1e-5, 1e-3, 0.5, 0)
    h = ctypes.c_void_p()
    assert lib.clt_create(ctypes.byref(g), ctypes.byref(p), None, 0, None, ctypes.byref(h)) == clt.CLT_EINVAL
    buf = np.zeros(1024)
    assert lib.clt_create(ctypes.byref(g), ctypes.byref(p), buf.ctypes.data, buf.nbytes, None, ctypes.byref(h)) \
        == clt.CLT_ENOMEM                                                   # too small
    assert lib.clt_set_state(None, None) == clt.CLT_EINVAL
    assert lib.clt_step(None, 1) == clt.CLT_EINVAL
    assert lib.clt_destroy(None) == clt.CLT_OK
    assert lib.clt_launch_count(None) == 0


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    g = clt.clt_grid(32, 16, 32, 2.0, 4.0, -1.0, 1.0, 0.0)
    p = clt.clt_params(5 / 3, 1e-5, 1e-5, 1e-5, 1e-5, 1e-3, 0.5, 0)
    nbytes = lib.clt_workspace_bytes(ctypes.byref(g))
    host = np.zeros(nbytes // 8 + 64)
    addr = (host.ctypes.data + 255) // 256 * 256
    h = ctypes.c_void_p()
    rc = lib.clt_create(ctypes.byref(g), ctypes.byref(p), addr, nbytes, None, ctypes.byref(h))
    assert rc in (clt.CLT_ECUDA, clt.CLT_ENOMEM) and not h.value            # host memory / no driver: refused
    with pytest.raises(RuntimeError):
        clt.Clt(32, 16, 32, 2.0, 4.0, -1.0, 1.0)

"""Host-side checks of libwpgrid.so that need no GPU: the library loads, exports every symbol
include/wpgrid.h declares, its host helpers agree with the oracle, and it refuses to compute
without a device (no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1905_03213_b200 import build as wbuild
from paper_1905_03213_b200 import wpgrid
from oracle import taper, wkernel

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    wbuild.build()
    return wpgrid.load()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "wpgrid.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(wpg_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(wpgrid.EXPORTS), declared ^ set(wpgrid.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    assert lib.wpg_version() >= 100


def test_struct_layouts_match_header():
    assert ctypes.sizeof(wpgrid.KDesc) == 56
    assert ctypes.sizeof(wpgrid.Stats) == 40
    assert ctypes.sizeof(wpgrid.BinInfo) == 48


def test_library_taper_matches_oracle(lib):
    nu = np.concatenate([np.linspace(-0.9999, 0.9999, 1001), [1.0, -1.0, 2.0]])
    got = wpgrid.taper(nu)
    assert np.max(np.abs(got - taper.psi(nu))) <= 1e-13
    assert got[-1] == 0.0 and got[-2] == 0.0 and got[-3] == 0.0


def test_ragged_support_matches_oracle(lib):
    for (Nw, w_max, N, cell) in [(128, 5.0e3, 8192, 1.0e-5), (16, 300.0, 512, 2e-4), (7, 1234.5, 1024, 8e-5)]:
        sup, off = wpgrid.ragged_support(Nw, w_max, N, cell, 8, 8, 32)
        assert np.array_equal(sup, wkernel.ragged_support(Nw, w_max, N, cell, 8, 32))
        assert off[0] == 0 and np.array_equal(np.diff(off), 64 * sup.astype(np.int64) ** 2)
    assert lib.wpg_wkernel_elems(16, 7, 8) == 16 * 64 * 49


def test_no_cpu_fallback_without_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = ctypes.c_void_p()
    rc = lib.wpg_create(ctypes.byref(h), 0, None)
    assert rc == wpgrid.ECUDA and not h.value
    assert b"no CPU fallback" in lib.wpg_last_error(None)
    with pytest.raises(wpgrid.WpgError):
        wpgrid.Context(0)


def test_workspace_planning_is_host_logic(lib):
    d, sup, off, uni = wpgrid.make_desc(32, 4700.0, 8, 8, 2048, 8.3e-5)
    n = lib.wpg_grid_workspace_bytes(None, 10_000_000, 1, ctypes.byref(d), wpgrid.F32)
    assert 10_000_000 * 16 < n < 10_000_000 * 19     # one 16 B record per visibility + 16.8 MB of bucket offsets
    # bad descriptors are refused (0 bytes)
    bad, *_ = wpgrid.make_desc(32, 4700.0, 7, 3, 2048, 8.3e-5)      # S*Q odd
    assert lib.wpg_grid_workspace_bytes(None, 1000, 1, ctypes.byref(bad), wpgrid.F32) == 0
    bad, *_ = wpgrid.make_desc(300, 4700.0, 8, 8, 2048, 8.3e-5)     # Nw > 256
    assert lib.wpg_grid_workspace_bytes(None, 1000, 1, ctypes.byref(bad), wpgrid.F32) == 0
    bad, *_ = wpgrid.make_desc(4, 10.0, 8, 8, 16384, 8.3e-5)        # N > 8192
    assert lib.wpg_grid_workspace_bytes(None, 1000, 1, ctypes.byref(bad), wpgrid.F32) == 0

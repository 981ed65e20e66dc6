"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol the header
declares; parameter validation and workspace sizing work; compute calls fail loudly without a device."""
import ctypes as C
import os
import re

import pytest

import workloads as W
from paper_2303_10785_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "meg6.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(meg6_[a-z0-9_]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol():
    L = B.lib()
    names = declared_symbols()
    assert set(names) == set(B.EXPORTS), (names, B.EXPORTS)
    for n in names:
        assert hasattr(L, n), n
    assert L.meg6_version() >= 1000


def test_workspace_bytes_and_validation():
    L = B.lib()
    wl = W.c1_vortex(n=32)
    p = B.make_params(wl["params"])
    nb = L.meg6_workspace_bytes(C.byref(p))
    # 22 geometry arrays of (n+20)^3, 9 interface arrays, 6 primitives, 10 state arrays: tens of MB
    assert 20e6 < nb < 200e6
    pv = B.make_params(dict(wl["params"], viscous=1, mu_ref=1e-3))
    assert L.meg6_workspace_bytes(C.byref(pv)) > nb
    bad = B.make_params(dict(wl["params"], ni=4))
    assert L.meg6_workspace_bytes(C.byref(bad)) == 0
    assert b"invalid" in L.meg6_last_error()
    mig4 = B.make_params(dict(wl["params"], scheme=1))
    assert L.meg6_workspace_bytes(C.byref(mig4)) > nb          # MIG4: line-solve arrays and pass scratch on top
    assert L.meg6_workspace_bytes(C.byref(B.make_params(dict(wl["params"], scheme=2)))) == 0


def test_no_silent_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(B.Meg6Error):
        B.Grid(W.c1_vortex(n=16))
    # raw ABI: grid_create must report MEG6_ECUDA (3), not succeed
    L = B.lib()
    p = B.make_params(W.c1_vortex(n=16)["params"])
    h = C.c_void_p()
    st = L.meg6_grid_create(C.byref(p), 256, 256, 256, None, None, None, 256, 1 << 40, None, C.byref(h))
    assert st == 3 and h.value is None


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2303_10785_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "meg6_oracle" not in txt and "import oracle" not in txt and "from oracle" not in txt, f

"""Host-side checks that need no GPU: the C-ABI library builds for sm_100a, loads, and exports
every function include/psc.h declares; argument validation that happens before any device work."""
import ctypes as C
import os
import re

import paper_1310_7866_b200 as psc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "psc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(psc_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    L = psc.lib()
    names = _declared()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), n
    assert sorted(psc.EXPORTS) == names


def test_version_and_strerror():
    assert "sm_100a" in psc.version()
    L = psc.lib()
    assert L.psc_strerror(0) == b"ok"
    for code in range(-9, 0):
        assert L.psc_strerror(code) not in (b"ok", b"unknown error")


def _params(**kw):
    p = psc.PscParams()
    n = kw.get("n", (1, 16, 16))
    for d in range(3):
        p.n[d] = n[d]
        p.dx[d] = 1.0
        p.block[d] = kw.get("block", (0, 0, 0))[d]
    p.ghost = kw.get("ghost", 2)
    p.dt = kw.get("dt", 0.35)
    p.order = kw.get("order", 1)
    p.n_species = 1
    q = (C.c_float * 1)(-1.0)
    m = (C.c_float * 1)(1.0)
    p.q = C.cast(q, C.POINTER(C.c_float))
    p.m = C.cast(m, C.POINTER(C.c_float))
    p._keep = (q, m)
    return p


def test_create_validates_before_touching_the_device():
    L = psc.lib()
    h = C.c_void_p()
    assert L.psc_create(None, C.byref(h)) == -1
    assert L.psc_create(C.byref(_params(order=3)), C.byref(h)) == -1
    bad = _params()
    bad.scheme = 2
    assert L.psc_create(C.byref(bad), C.byref(h)) == -1
    assert L.psc_create(C.byref(_params(ghost=1)), C.byref(h)) == -1
    assert L.psc_create(C.byref(_params(n=(1, 3, 16))), C.byref(h)) == -1
    assert L.psc_create(C.byref(_params(dt=0.6)), C.byref(h)) == -4          # PSC_ERR_CFL
    assert L.psc_create(C.byref(_params(block=(1, 5, 4))), C.byref(h)) == -1  # must divide n
    assert h.value is None


def test_no_cpu_fallback_without_a_device():
    """without a CUDA device a valid psc_create fails with PSC_ERR_CUDA instead of falling back"""
    import torch

    if torch.cuda.is_available():
        return
    h = C.c_void_p()
    assert psc.lib().psc_create(C.byref(_params()), C.byref(h)) == -6

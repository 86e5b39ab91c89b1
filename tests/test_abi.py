"""Host-side checks of the C-ABI boundary that need no GPU: the library loads, exports every
symbol include/ok.h declares, sizes follow SURVEY.md 8(a), bad arguments are rejected."""
import ctypes as C
import os
import re

import pytest

from paper_1311_5029_b200 import binding as B
from paper_1311_5029_b200 import build as okbuild
from paper_1311_5029_b200 import inputs as I

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    okbuild.build()
    return B.lib()


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "ok.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(ok_[a-zA-Z_0-9]+)\s*\(", txt)))


def test_every_declared_symbol_is_exported_and_bound(lib):
    names = declared_symbols()
    assert {"ok_precalc_W", "ok_dirac_apply", "ok_bicgstab"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
        assert n in B.EXPORTS, f"{n} declared in ok.h but not bound in binding.py"
    assert set(B.EXPORTS) == set(names)


def test_struct_layout_matches_header():
    # 10 int32 + 12 double + storage, reserved_ (2 int32), no padding surprises: 40 + 96 + 8 = 144 bytes
    assert C.sizeof(B.ok_params) == 144
    assert B.ok_params.storage.offset == 136


def test_sizes(lib):
    p = B.make_params(I.make_params((20, 20, 20, 64), 0.1, 0.95), B.OK_FP32)
    V = 20 ** 3 * 64
    assert B.ok_W_bytes(p) == 1024 + V * 27 * 144 * 8          # 31 104 B/site fp32
    assert B.ok_vec_bytes(p) == V * 96
    p64 = B.make_params(I.make_params((4, 4, 4, 8), 0.1, 0.95), B.OK_FP64)
    assert B.ok_W_bytes(p64) == 1024 + 512 * 27 * 144 * 16
    # ragged lattice: 4*3*3*2 = 72 sites -> 3 blocks of 32
    pr = B.make_params(I.make_params((4, 3, 3, 2), 0.1, 0.95), B.OK_FP64)
    assert B.ok_vec_bytes(pr) == 96 * 12 * 16
    assert B.ok_work_bytes(pr) > 0
    pm = B.make_params(I.make_params((4, 4, 4, 8), 0.1, 0.95), B.OK_FP32, nrhs=12)
    assert B.ok_vec_bytes(pm) == 256 + 2 * 512 * 12 * 12 * 8     # header + fp32 records + tensor-core operand records
    # reduced storage formats: 260 resp. 132 colour blocks of 9 complex per site
    pb = B.make_params(I.make_params((20, 20, 20, 64), 0.1, 0.95), B.OK_FP32, storage=B.OK_W_BLOCK)
    assert B.ok_W_bytes(pb) == 1024 + V * 260 * 9 * 8            # 18 720 B/site
    pds = B.make_params(I.make_params((20, 20, 20, 64), 0.1, 0.95), B.OK_FP32, storage=B.OK_W_DS)
    assert B.ok_W_bytes(pds) == 1024 + V * 132 * 9 * 8           # 9 504 B/site
    assert B.ok_W_bytes(B.make_params(I.make_params((4, 4, 4, 8), 0.1, 0.95), B.OK_FP32, nrhs=12, storage=B.OK_W_DS)) == 0


def test_invalid_params_rejected(lib):
    bad = B.make_params(I.make_params((1, 4, 4, 4), 0.1, 0.95), B.OK_FP64)
    assert B.ok_W_bytes(bad) == 0 and B.ok_vec_bytes(bad) == 0
    bad = B.make_params(I.make_params((4, 4, 4, 4), 0.1, 0.95), 7)
    assert B.ok_W_bytes(bad) == 0
    bad = B.make_params(I.make_params((4, 4, 4, 4), 0.1, 0.95), B.OK_FP64, nrhs=12)   # multi-RHS is fp32 only
    assert B.ok_W_bytes(bad) == 0
    bad = B.make_params(I.make_params((4, 4, 4, 4), 0.1, 0.95, bc=(1, 1, 0, -1)), B.OK_FP64)
    assert B.ok_W_bytes(bad) == 0
    good = B.make_params(I.make_params((4, 4, 4, 4), 0.1, 0.95), B.OK_FP64)
    # null / misaligned pointers -> OK_EINVAL, before any CUDA call
    assert lib.ok_pack_spinor(C.byref(good), None, None) == -1
    assert lib.ok_precalc_W(8, C.byref(good), 24) == -1
    assert lib.ok_dirac_apply(None, None, None) == -1
    assert lib.ok_set_workspace(12, 100) == -1
    it, rs = C.c_int(), C.c_double()
    assert lib.ok_bicgstab(None, None, None, 1e-6, 10, C.byref(it), C.byref(rs)) == -1
    assert "invalid" in B.ok_strerror(-1)
    assert "okdirac" in B.ok_version()


def test_missing_library_fails_loudly(monkeypatch):
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "_LIB_PATH", "/nonexistent/libokdirac.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        B.lib()

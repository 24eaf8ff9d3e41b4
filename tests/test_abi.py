"""CPU-only checks of the C-ABI boundary (include/letkf.h): the library builds for sm_100a,
loads, exports every declared symbol, and validates arguments before touching a device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2308_03310_b200 import build, letkf
    build.build()
    return letkf.load()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "letkf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(letkf_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_entry_points():
    names = declared_functions()
    for must in ("letkf_syev_batched", "letkf_analysis_batched"):
        assert must in names


def test_every_declared_symbol_is_exported(lib):
    from paper_2308_03310_b200 import letkf
    names = declared_functions()
    assert sorted(letkf.EXPORTS) == names
    for n in names:
        assert hasattr(lib, n), n


def test_version_and_status_string(lib):
    assert lib.letkf_version() == 100
    assert lib.letkf_status_string(0) == b"ok"
    assert b"argument 3" in lib.letkf_status_string(-3)


def test_argument_validation_needs_no_device(lib):
    null = ctypes.c_void_p(0)
    fake = ctypes.c_void_p(0x1000)          # aligned, never dereferenced
    odd = ctypes.c_void_p(0x1008)           # misaligned
    syev = lib.letkf_syev_batched
    assert syev(fake, 0, 4, fake, fake, null, null, 0, null) == -2        # M < 1
    assert syev(fake, 257, 4, fake, fake, null, null, 0, null) == -2      # M > LETKF_MAX_M
    assert syev(fake, 8, -1, fake, fake, null, null, 0, null) == -3       # batch < 0
    assert syev(null, 8, 0, null, null, null, null, 0, null) == 0         # batch == 0: no-op
    assert syev(null, 8, 4, fake, fake, null, null, 0, null) == -1        # A NULL
    assert syev(odd, 8, 4, fake, fake, null, null, 0, null) == -1         # A misaligned
    assert syev(fake, 8, 4, null, fake, null, null, 0, null) == -4        # w NULL
    assert syev(fake, 8, 4, fake, null, null, null, 0, null) == -5        # V NULL
    assert syev(fake, 8, 4, fake, fake, null, fake, 16, null) == -7       # workspace too small
    ana = lib.letkf_analysis_batched
    args = lambda **k: [k.get("Yb", fake), fake, fake, k.get("Xb", fake), k.get("M", 8), k.get("p", 3),
                        k.get("ns", 2), k.get("batch", 4), k.get("rho", 1.1), k.get("Xa", fake),
                        null, null, null, null, 0, null]
    assert ana(*args(M=0)) == -5
    assert ana(*args(M=1)) == -5
    assert ana(*args(p=-1)) == -6
    assert ana(*args(ns=0)) == -7
    assert ana(*args(batch=-2)) == -8
    assert ana(*args(rho=0.0)) == -9
    assert ana(*args(batch=0)) == 0
    assert ana(*args(Yb=null)) == -1
    assert ana(*args(Xb=null)) == -4
    assert ana(*args(Xa=null)) == -10


def test_workspace_sizes(lib):
    assert lib.letkf_syev_workspace_bytes(64, 0) == 0
    a = lib.letkf_syev_workspace_bytes(64, 1024)
    b = lib.letkf_syev_workspace_bytes(64, 16384)
    assert 0 < a <= b < (3 << 30)
    assert lib.letkf_analysis_workspace_bytes(64, 98, 9, 1024) > a


def test_binding_fails_loudly_without_library(monkeypatch, tmp_path):
    from paper_2308_03310_b200 import letkf
    monkeypatch.setattr(letkf, "_lib", None)
    monkeypatch.setattr(letkf, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(letkf.LetkfError):
        letkf.load()


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2308_03310_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "oracle.h" not in src and "liboracle" not in src, f


def test_host_entry_points_validate_before_touching_a_device(lib):
    null = ctypes.c_void_p(0)
    fake = ctypes.c_void_p(0x1000)
    hs = lib.letkf_syev_batched_host
    assert hs(fake, 0, 4, fake, fake, null) == -2
    assert hs(fake, 8, -1, fake, fake, null) == -3
    assert hs(null, 8, 0, null, null, null) == 0
    assert hs(null, 8, 4, fake, fake, null) == -1
    assert hs(fake, 8, 4, null, fake, null) == -4
    assert hs(fake, 8, 4, fake, null, null) == -5
    ha = lib.letkf_analysis_batched_host
    assert ha(fake, fake, fake, fake, 1, 3, 2, 4, 1.1, fake, null, null, null) == -5
    assert ha(fake, fake, fake, fake, 8, -1, 2, 4, 1.1, fake, null, null, null) == -6
    assert ha(fake, fake, fake, fake, 8, 3, 0, 4, 1.1, fake, null, null, null) == -7
    assert ha(fake, fake, fake, fake, 8, 3, 2, 4, 0.0, fake, null, null, null) == -9
    assert ha(null, fake, fake, fake, 8, 3, 2, 4, 1.1, fake, null, null, null) == -1
    assert ha(fake, fake, fake, null, 8, 3, 2, 4, 1.1, fake, null, null, null) == -4
    assert ha(fake, fake, fake, fake, 8, 3, 2, 4, 1.1, null, null, null, null) == -10
    assert ha(null, null, null, null, 8, 3, 2, 0, 1.1, null, null, null, null) == 0


def test_grid_entry_points_validate_before_touching_a_device(lib):
    null = ctypes.c_void_p(0)
    fake = ctypes.c_void_p(0x1000)
    g = lib.letkf_analysis_grid
    ok = dict(M=8, V=2, Ny=4, Nx=4, ns=2, hw=1, kind=0, L=2.0, sig=0.1, rho=1.1)

    def call(Yf=fake, yo=fake, Xb=fake, Xa=fake, **k):
        a = dict(ok, **k)
        return g(Yf, yo, null, Xb, a["M"], a["V"], a["Ny"], a["Nx"], a["ns"], a["hw"], a["kind"], a["L"], a["sig"],
                 a["rho"], Xa, null, null, null, 0, null)
    assert call(M=1) == -5 and call(V=0) == -6 and call(Ny=0) == -7 and call(Nx=0) == -8
    assert call(ns=0) == -9 and call(hw=-1) == -10 and call(kind=2) == -11 and call(L=0.0) == -12
    assert call(sig=0.0) == -13 and call(rho=-1.0) == -14
    assert call(Yf=null) == -1 and call(yo=null) == -2 and call(Xb=null) == -4 and call(Xa=null) == -15
    assert lib.letkf_analysis_grid_workspace_bytes(64, 2, 128, 128, 3, 9) > 0
    assert lib.letkf_analysis_grid_workspace_bytes(1, 2, 128, 128, 3, 9) == 0
    h = lib.letkf_analysis_grid_host
    assert h(fake, fake, null, fake, 1, 2, 4, 4, 2, 1, 0, 2.0, 0.1, 1.1, fake, null, null) == -5
    assert h(null, fake, null, fake, 8, 2, 4, 4, 2, 1, 0, 2.0, 0.1, 1.1, fake, null, null) == -1

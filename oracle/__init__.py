"""ctypes loader for the CPU ORACLE (oracle/oracle.c).

TEST INFRASTRUCTURE -- importable only from tests/, ``__graft_entry__.smoke()`` and
``bench.py``'s cpu_baseline / ``--impl reference`` legs.  The product package
(``paper_2308_03310_b200``) never imports this module and this module never imports it.

The functions mirror oracle.h one to one (numpy arrays in, numpy arrays out); the
arithmetic lives in C, see oracle.c / jacobi_impl.inc for the citations.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = [os.path.join(_HERE, f) for f in ("oracle.c", "jacobi_impl.inc", "oracle.h")]
_lib = None


def build(force=False):
    """Compile oracle.c -> liboracle.so with gcc (no fast-math, no FMA contraction)."""
    if not force and os.path.exists(_SO) and all(
            os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC):
        return _SO
    cmd = ["gcc", "-std=c99", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
           "-o", _SO, os.path.join(_HERE, "oracle.c"), "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        dp, ip, ci, cd = (ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int),
                          ctypes.c_int, ctypes.c_double)
        lib.oracle_syev.argtypes = [dp, ci, dp, dp]
        lib.oracle_syev.restype = ci
        lib.oracle_syev_ld.argtypes = [dp, ci, dp, dp]
        lib.oracle_syev_ld.restype = ci
        lib.oracle_syev_batched.argtypes = [dp, ci, ci, dp, dp, ip, ci]
        lib.oracle_syev_batched.restype = ci
        lib.oracle_letkf_analysis_batched.argtypes = [dp, dp, dp, dp, ci, ci, ci, ci, cd,
                                                      dp, dp, dp, ip, ci]
        lib.oracle_letkf_analysis_batched.restype = ci
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _c(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def syev(A, long_double=False):
    """EVD of one symmetric matrix (lower triangle read). Returns (w, V, sweeps)."""
    lib = _load()
    A = _c(A)
    M = A.shape[-1]
    assert A.shape == (M, M)
    w = np.empty(M)
    V = np.empty((M, M))
    fn = lib.oracle_syev_ld if long_double else lib.oracle_syev
    sweeps = fn(_dp(A), M, _dp(w), _dp(V))
    return w, V, sweeps


def syev_batched(A, nthreads=0):
    """EVD of A[batch][M][M]. Returns (w, V, info, threads_used)."""
    lib = _load()
    A = _c(A)
    batch, M, M2 = A.shape
    assert M == M2
    w = np.empty((batch, M))
    V = np.empty((batch, M, M))
    info = np.zeros(batch, dtype=np.int32)
    nt = lib.oracle_syev_batched(_dp(A), M, batch, _dp(w), _dp(V),
                                 info.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), nthreads)
    return w, V, info, nt


def letkf_analysis_batched(Yb, d, rinv_loc, Xb, rho, nthreads=0, want_W=True):
    """Local analysis for every grid point. Returns dict(Xa, W, wbar, info, threads)."""
    lib = _load()
    Yb, d, rinv_loc, Xb = _c(Yb), _c(d), _c(rinv_loc), _c(Xb)
    batch, p, M = Yb.shape
    ns = Xb.shape[1]
    assert d.shape == (batch, p) and rinv_loc.shape == (batch, p)
    assert Xb.shape == (batch, ns, M)
    Xa = np.empty((batch, ns, M))
    W = np.empty((batch, M, M)) if want_W else None
    wbar = np.empty((batch, M))
    info = np.zeros(batch, dtype=np.int32)
    nt = lib.oracle_letkf_analysis_batched(
        _dp(Yb), _dp(d), _dp(rinv_loc), _dp(Xb), M, p, ns, batch, float(rho),
        _dp(Xa), _dp(W) if want_W else None, _dp(wbar),
        info.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), nthreads)
    return dict(Xa=Xa, W=W, wbar=wbar, info=info, threads=nt)


def localisation(loc_kind, L, dist):
    lib = _load()
    lib.oracle_localisation.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.c_double]
    lib.oracle_localisation.restype = ctypes.c_double
    return lib.oracle_localisation(int(loc_kind), float(L), float(dist))


def letkf_analysis_grid(Yf, yo, Xb, hw, loc_kind, L, sigma_o, rho, mask=None, nthreads=0):
    """Grid form: Yf[V][Ny][Nx][M], yo[V][Ny][Nx], Xb[Ny*Nx][nstate][M] -> dict(Xa, wbar, info)."""
    lib = _load()
    Yf, yo, Xb = _c(Yf), _c(yo), _c(Xb)
    V, Ny, Nx, M = Yf.shape
    ns = Xb.shape[1]
    assert yo.shape == (V, Ny, Nx) and Xb.shape == (Ny * Nx, ns, M)
    mk = None
    if mask is not None:
        mk = np.ascontiguousarray(mask, dtype=np.uint8)
        assert mk.shape == (Ny, Nx)
    Xa = np.empty_like(Xb)
    wbar = np.empty((Ny * Nx, M))
    info = np.zeros(Ny * Nx, dtype=np.int32)
    lib.oracle_letkf_analysis_grid.argtypes = [
        ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
        ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
        ctypes.c_double, ctypes.c_double, ctypes.c_double,
        ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
    lib.oracle_letkf_analysis_grid.restype = ctypes.c_int
    nt = lib.oracle_letkf_analysis_grid(
        Yf.ctypes.data, yo.ctypes.data, mk.ctypes.data if mk is not None else None, Xb.ctypes.data,
        M, V, Ny, Nx, ns, int(hw), int(loc_kind), float(L), float(sigma_o), float(rho),
        Xa.ctypes.data, wbar.ctypes.data, info.ctypes.data, nthreads)
    return dict(Xa=Xa, wbar=wbar, info=info, threads=nt)


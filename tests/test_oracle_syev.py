"""Pins for oracle_syev (CPU only).  Each test checks the oracle against something the
mathematics fixes, not against itself: SURVEY.md section 8(c) pins P-1 ... P-6.

The operation pinned is the "EVD of Q" of PAPER.md:142.
"""
import itertools
import math

import numpy as np
import pytest

from harness import workloads as wl

EPS = np.finfo(np.float64).eps


def _check_evd(A, w, V, tol=1e-13):
    M = A.shape[0]
    nrm = np.abs(w).max() if M else 1.0
    assert np.all(np.diff(w) >= 0), "eigenvalues must be ascending"
    R = A @ V - V * w[None, :]
    assert np.linalg.norm(R) <= tol * max(np.linalg.norm(A), 1e-300) * M
    assert np.abs(V.T @ V - np.eye(M)).max() <= tol * M
    return nrm


# P-1 -------------------------------------------------------------------------------------
def test_known_spectrum_config1(oracle):
    """A = Q diag(lam) Q^T by construction (BASELINE.json config 1): eigenvalues are lam."""
    A, lam = wl.known_spectrum(batch=64, M=32)
    w, V, info, _ = oracle.syev_batched(A)
    assert not info.any()
    # building A in fp64 with 32 reflectors perturbs the spectrum by a few eps*||A||
    assert np.abs(w - lam).max() <= 2e-13 * 100.0
    for b in range(0, 64, 7):
        _check_evd(A[b], w[b], V[b])


# P-2 -------------------------------------------------------------------------------------
@pytest.mark.parametrize("a,b,c", [(2.0, 1.0, 3.0), (1.0, 0.0, 1.0), (-4.0, 2.5, 7.0),
                                   (5.0, 1e-9, 5.0), (0.0, 3.0, 0.0), (1e8, 1.0, -1e8)])
def test_2x2_closed_form(oracle, a, b, c):
    A = np.array([[a, b], [b, c]])
    w, V, _ = oracle.syev(A)
    mid, rad = 0.5 * (a + c), math.hypot(0.5 * (a - c), b)
    scale = max(abs(mid) + rad, 1e-300)
    assert abs(w[0] - (mid - rad)) <= 4 * EPS * scale
    assert abs(w[1] - (mid + rad)) <= 4 * EPS * scale
    if b != 0.0:
        # eigenvector of the LARGER eigenvalue makes angle phi = atan2(2b, a-c)/2 with e_1
        phi = 0.5 * math.atan2(2 * b, a - c)
        v = np.array([math.cos(phi), math.sin(phi)])
        assert abs(abs(v @ V[:, 1]) - 1.0) <= 64 * EPS
    _check_evd(A, w, V)


# P-3 -------------------------------------------------------------------------------------
@pytest.mark.parametrize("M", [1, 2, 3, 5, 16, 33, 64])
@pytest.mark.parametrize("a,b", [(0.0, 1.0), (2.0, -1.0), (-3.0, 0.5)])
def test_tridiagonal_toeplitz(oracle, M, a, b):
    """tridiag(b,a,b): lam_k = a + 2 b cos(k pi/(M+1)), v_k(j) = sqrt(2/(M+1)) sin(jk pi/(M+1))."""
    A = wl.toeplitz_tridiagonal(M, a, b)
    w, V, sweeps = oracle.syev(A)
    assert sweeps >= 0
    k = np.arange(1, M + 1)
    lam = a + 2 * b * np.cos(k * math.pi / (M + 1))
    order = np.argsort(lam)
    assert np.abs(w - lam[order]).max() <= 40 * EPS * (abs(a) + 2 * abs(b))
    j = np.arange(1, M + 1)
    Vexact = math.sqrt(2.0 / (M + 1)) * np.sin(np.outer(j, k[order]) * math.pi / (M + 1))
    overlap = np.abs(np.sum(Vexact * V, axis=0))   # |<v_exact, v>| per eigenpair (gaps are O(1/M^2))
    assert np.abs(overlap - 1.0).max() <= 1e-11
    _check_evd(A, w, V)


# P-4 -------------------------------------------------------------------------------------
@pytest.mark.parametrize("M", [1, 2, 3, 7, 16, 31, 48, 64, 96])
def test_invariants_random_symmetric(oracle, M):
    rng = np.random.Generator(np.random.Philox(key=1000 + M))
    B = rng.standard_normal((M, M))
    A = 0.5 * (B + B.T) * 3.0 - 1.0
    w, V, _ = oracle.syev(A)
    nrm = _check_evd(A, w, V)
    assert abs(np.trace(A) - w.sum()) <= 8 * EPS * M * nrm
    assert abs(np.sum(A * A) - np.sum(w * w)) <= 16 * EPS * M * nrm * nrm


def test_reads_lower_triangle_only(oracle):
    rng = np.random.Generator(np.random.Philox(key=77))
    B = rng.standard_normal((9, 9))
    A = 0.5 * (B + B.T)
    junk = np.tril(A) + np.triu(rng.standard_normal((9, 9)), 1) * 1e3
    w0, _, _ = oracle.syev(A)
    w1, _, _ = oracle.syev(junk)
    assert np.array_equal(w0, w1)


def test_spd_letkf_shaped_positive_and_cluster(oracle):
    """(M-1)/rho I + low rank: (M-p)-fold eigenvalue at exactly (M-1)/rho."""
    M, p = 24, 5
    A = wl.letkf_shaped(3, M, p, config_index=901)
    for b in range(3):
        w, V, _ = oracle.syev(A[b])
        _check_evd(A[b], w, V)
        base = (M - 1) / wl.RHO
        # rows of Yb are centred -> rank <= min(p, M-1); here p < M-1
        assert np.abs(w[: M - p] - base).max() <= 1e-12 * w.max()
        assert w[M - p] > base * (1 + 1e-6)


# P-5 -------------------------------------------------------------------------------------
def _det_minors(B):
    """Laplace expansion along the first row (explicit minors), long double."""
    n = B.shape[0]
    if n == 1:
        return B[0, 0]
    if n == 2:
        return B[0, 0] * B[1, 1] - B[0, 1] * B[1, 0]
    tot = np.longdouble(0)
    for j in range(n):
        minor = np.delete(np.delete(B, 0, axis=0), j, axis=1)
        tot += (-1) ** j * B[0, j] * _det_minors(minor)
    return tot


@pytest.mark.parametrize("M", [2, 3, 4])
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_characteristic_polynomial_bruteforce(oracle, M, seed):
    rng = np.random.Generator(np.random.Philox(key=500 + 10 * M + seed))
    # well separated spectrum so that a grid scan isolates every root
    lam = np.sort(rng.uniform(-5, 5, M))
    while M > 1 and np.diff(lam).min() < 0.3:
        lam = np.sort(rng.uniform(-5, 5, M))
    Q, _ = np.linalg.qr(rng.standard_normal((M, M)))
    A = (Q * lam) @ Q.T
    A = 0.5 * (A + A.T)
    AL = A.astype(np.longdouble)
    I = np.eye(M, dtype=np.longdouble)

    def charpoly(x):
        return _det_minors(AL - np.longdouble(x) * I)

    grid = np.linspace(-7, 7, 1401)
    vals = np.array([charpoly(x) for x in grid])
    roots = []
    for i in range(len(grid) - 1):
        if vals[i] == 0:
            roots.append(grid[i])
        elif vals[i] * vals[i + 1] < 0:
            lo, hi, flo = np.longdouble(grid[i]), np.longdouble(grid[i + 1]), vals[i]
            for _ in range(80):
                mid = (lo + hi) / 2
                fm = charpoly(mid)
                if (fm < 0) == (flo < 0):
                    lo, flo = mid, fm
                else:
                    hi = mid
            roots.append(float((lo + hi) / 2))
    assert len(roots) == M
    w, V, _ = oracle.syev(A)
    assert np.abs(w - np.array(roots)).max() <= 1e-13 * 7
    _check_evd(A, w, V)


# P-6 (secondary library cross-check) ------------------------------------------------------
@pytest.mark.parametrize("name", ["config2", "config3"])
def test_against_lapack_eigh(oracle, name):
    A = getattr(wl, name)(batch=8)
    w, V, info, _ = oracle.syev_batched(A)
    wl_, _ = np.linalg.eigh(A)
    assert not info.any()
    assert np.abs(w - wl_).max() <= 1e-13 * np.abs(wl_).max()
    for b in range(8):
        _check_evd(A[b], w[b], V[b])


def test_long_double_referee_agrees(oracle):
    A = wl.config3(batch=2)[1]
    w, V, _ = oracle.syev(A)
    wr, Vr, _ = oracle.syev(A, long_double=True)
    assert np.abs(w - wr).max() <= 1e-13 * wr.max()
    _check_evd(A, wr, Vr, tol=2e-15)


def test_degenerate_inputs(oracle):
    # A = c I: nothing to rotate, V = I
    w, V, sweeps = oracle.syev(4.0 * np.eye(6))
    assert sweeps == 0 and np.array_equal(w, np.full(6, 4.0)) and np.array_equal(V, np.eye(6))
    # zero matrix
    w, V, _ = oracle.syev(np.zeros((5, 5)))
    assert np.array_equal(w, np.zeros(5)) and np.array_equal(V, np.eye(5))
    # M = 1
    w, V, _ = oracle.syev(np.array([[-2.5]]))
    assert w[0] == -2.5 and V[0, 0] == 1.0
    # batch = 0
    w, V, info, _ = oracle.syev_batched(np.zeros((0, 4, 4)))
    assert w.shape == (0, 4)

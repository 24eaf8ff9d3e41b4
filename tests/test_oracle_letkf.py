"""Pins for oracle_letkf_analysis_batched (CPU only): SURVEY.md section 8(c) pins P-7 ... P-11.

The operation pinned is the local problem of one grid point, Eq.13-19,
tied back to the Kalman filter it must reproduce, Eq.6-8 and Eq.12.
"""
import math

import numpy as np
import pytest

from harness import workloads as wl


def gauss_solve(Ain, Bin):
    """Gaussian elimination with partial pivoting, written out (no library solve)."""
    A = np.array(Ain, dtype=np.float64)
    B = np.array(Bin, dtype=np.float64).reshape(A.shape[0], -1)
    n = A.shape[0]
    for k in range(n):
        piv = k + int(np.argmax(np.abs(A[k:, k])))
        if piv != k:
            A[[k, piv]] = A[[piv, k]]
            B[[k, piv]] = B[[piv, k]]
        for i in range(k + 1, n):
            f = A[i, k] / A[k, k]
            A[i, k:] -= f * A[k, k:]
            B[i] -= f * B[k]
    X = np.zeros_like(B)
    for i in range(n - 1, -1, -1):
        X[i] = (B[i] - A[i, i + 1:] @ X[i + 1:]) / A[i, i]
    return X


def _run(oracle, inp, **kw):
    return oracle.letkf_analysis_batched(inp["Yb"], inp["d"], inp["rinv_loc"], inp["Xb"],
                                         kw.get("rho", inp["rho"]))


# P-7 -------------------------------------------------------------------------------------
@pytest.mark.parametrize("M,p,ns,rho", [(64, 98, 9, 1.1), (16, 5, 9, 1.0), (8, 12, 3, 1.3),
                                        (5, 1, 1, 1.0), (32, 48, 9, 1.1)])
def test_kalman_filter_equivalence(oracle, M, p, ns, rho):
    """With a LINEAR observation operator, Yb = H dX, the ensemble-space update Eq.13-17
    must reproduce the model-space Kalman filter Eq.6-8 with P^f = rho dX dX^T/(M-1) (Eq.12):
       mean(Xa) = xbar + K d,   cov(Xa) = (I - K H) P^f,   K = P^f H^T (H P^f H^T + R)^-1."""
    rng = np.random.Generator(np.random.Philox(key=4242 + M * 7 + p))
    H = rng.standard_normal((p, ns))
    Xb = 0.3 + 0.2 * rng.standard_normal((ns, M))
    xbar = Xb.mean(axis=1)
    dX = Xb - xbar[:, None]
    Yb = H @ dX
    d = rng.standard_normal(p)
    r = rng.uniform(0.5, 20.0, p)
    out = oracle.letkf_analysis_batched(Yb[None], d[None], r[None], Xb[None], rho)
    Xa = out["Xa"][0]

    Pf = rho * dX @ dX.T / (M - 1)
    S = H @ Pf @ H.T + np.diag(1.0 / r)
    K = gauss_solve(S.T, (Pf @ H.T).T).T          # K S = Pf H^T
    mean_kf = xbar + K @ d
    Pa_kf = (np.eye(ns) - K @ H) @ Pf
    mean_a = Xa.mean(axis=1)
    dXa = Xa - mean_a[:, None]
    Pa = dXa @ dXa.T / (M - 1)
    assert np.abs(mean_a - mean_kf).max() <= 2e-12 * max(1.0, np.abs(mean_kf).max())
    assert np.abs(Pa - Pa_kf).max() <= 2e-12 * max(np.abs(Pf).max(), 1e-30)


def test_scalar_kalman_closed_form(oracle):
    """ns = p = 1: K = rho Pf h / (rho Pf h^2 + R), Pa = (1 - K h) rho Pf."""
    M, rho, h, rinv, dval = 10, 1.2, 0.7, 4.0, 0.35
    rng = np.random.Generator(np.random.Philox(key=99))
    x = rng.standard_normal(M)
    dx = x - x.mean()
    out = oracle.letkf_analysis_batched((h * dx)[None, None, :], np.array([[dval]]),
                                        np.array([[rinv]]), x[None, None, :], rho)
    Xa = out["Xa"][0, 0]
    Pf = rho * (dx @ dx) / (M - 1)
    K = Pf * h / (Pf * h * h + 1.0 / rinv)
    assert abs(Xa.mean() - (x.mean() + K * dval)) <= 1e-13
    assert abs(np.var(Xa, ddof=1) - (1 - K * h) * Pf) <= 1e-13


# P-8 -------------------------------------------------------------------------------------
@pytest.mark.parametrize("M,p", [(64, 98), (48, 49), (64, 3), (64, 48), (17, 30)])
def test_structural_identities(oracle, M, p):
    inp = wl.analysis_inputs(batch=3, M=M, p=p, config_index=300 + p)
    out = _run(oracle, inp)
    rho = inp["rho"]
    for b in range(3):
        Yb, r, d, Xb = inp["Yb"][b], inp["rinv_loc"][b], inp["d"][b], inp["Xb"][b]
        W, wbar, Xa = out["W"][b], out["wbar"][b], out["Xa"][b]
        A = (M - 1) / rho * np.eye(M) + (Yb.T * r) @ Yb
        g = Yb.T @ (r * d)
        nA = np.linalg.norm(A, 2)
        assert np.abs(W - W.T).max() <= 1e-14 * np.abs(W).max()
        assert np.abs(W @ A @ W - (M - 1) * np.eye(M)).max() <= 1e-12 * (M - 1)
        assert np.abs(A @ wbar - g).max() <= 1e-13 * max(nA * np.abs(wbar).max(), 1e-300)
        # rows of Yb centred => A 1 = ((M-1)/rho) 1 => W 1 = sqrt(rho) 1
        assert np.abs(W @ np.ones(M) - math.sqrt(rho)).max() <= 1e-13
        xbar = Xb.mean(axis=1, keepdims=True)
        dX = Xb - xbar
        assert np.abs(Xa.mean(axis=1) - (xbar[:, 0] + dX @ wbar)).max() <= 1e-14
        dXa = Xa - Xa.mean(axis=1, keepdims=True)
        ref = (M - 1) * dX @ gauss_solve(A, dX.T)
        assert np.abs(dXa @ dXa.T - ref).max() <= 1e-12 * np.abs(ref).max()
        # eigenvalues of W are sqrt((M-1)/lam) > 0: principal root (reading G2)
        assert np.linalg.eigvalsh(W).min() > 0


# P-9 -------------------------------------------------------------------------------------
@pytest.mark.parametrize("rho", [1.0, 1.1, 2.0])
def test_no_observations_closed_form(oracle, rho):
    """p = 0 or r = 0: A = ((M-1)/rho) I, W = sqrt(rho) I, wbar = 0, Xa = xbar + sqrt(rho) dX."""
    M, ns = 12, 4
    inp = wl.analysis_inputs(batch=2, M=M, p=6, nstate=ns, config_index=77)
    for variant in ("p0", "r0"):
        if variant == "p0":
            out = oracle.letkf_analysis_batched(np.zeros((2, 0, M)), np.zeros((2, 0)),
                                                np.zeros((2, 0)), inp["Xb"], rho)
        else:
            out = oracle.letkf_analysis_batched(inp["Yb"], inp["d"], 0 * inp["rinv_loc"],
                                                inp["Xb"], rho)
        xbar = inp["Xb"].mean(axis=2, keepdims=True)
        expect = xbar + math.sqrt(rho) * (inp["Xb"] - xbar)
        assert np.abs(out["Xa"] - expect).max() <= 4e-16
        assert np.abs(out["W"] - math.sqrt(rho) * np.eye(M)).max() <= 4e-16
        assert np.array_equal(out["wbar"], np.zeros((2, M)))
        if rho == 1.0:
            assert np.abs(out["Xa"] - inp["Xb"]).max() <= 3e-17 + 2.3e-16 * np.abs(inp["Xb"]).max()


def test_two_member_closed_form(oracle):
    """M = 2: centred rows are (y, -y); A has eigenpairs (1/rho, (1,1)/sqrt2) and
    (1/rho + 2 sum r y^2, (1,-1)/sqrt2); W and wbar follow in closed form."""
    rho = 1.1
    y = np.array([0.3, -1.2, 0.8])
    r = np.array([2.0, 0.5, 4.0])
    d = np.array([0.1, -0.4, 0.25])
    Yb = np.stack([y, -y], axis=1)                      # [p][2]
    Xb = np.array([[1.0, 3.0], [-2.0, 0.5]])
    out = oracle.letkf_analysis_batched(Yb[None], d[None], r[None], Xb[None], rho)
    l1, l2 = 1.0 / rho, 1.0 / rho + 2.0 * np.sum(r * y * y)
    u1 = np.array([1.0, 1.0]) / math.sqrt(2)
    u2 = np.array([1.0, -1.0]) / math.sqrt(2)
    W = np.outer(u1, u1) / math.sqrt(l1) + np.outer(u2, u2) / math.sqrt(l2)   # sqrt(M-1)=1
    g = Yb.T @ (r * d)
    wbar = u1 * (u1 @ g) / l1 + u2 * (u2 @ g) / l2
    assert np.abs(out["W"][0] - W).max() <= 1e-15
    assert np.abs(out["wbar"][0] - wbar).max() <= 1e-15
    xbar = Xb.mean(axis=1, keepdims=True)
    Xa = xbar + (Xb - xbar) @ (wbar[:, None] + W)
    assert np.abs(out["Xa"][0] - Xa).max() <= 1e-15


def test_zero_innovation_gives_zero_mean_weights(oracle):
    inp = wl.analysis_inputs(batch=2, M=20, p=15, config_index=55)
    out = oracle.letkf_analysis_batched(inp["Yb"], 0 * inp["d"], inp["rinv_loc"], inp["Xb"], 1.1)
    assert np.array_equal(out["wbar"], np.zeros((2, 20)))


def test_rho_one_is_eq17(oracle):
    """rho = 1 must give Q = (M-1) I + dY^T R^-1 dY exactly as printed (Eq.17)."""
    M, p = 10, 7
    inp = wl.analysis_inputs(batch=1, M=M, p=p, config_index=56)
    out = oracle.letkf_analysis_batched(inp["Yb"], inp["d"], inp["rinv_loc"], inp["Xb"], 1.0)
    Q = (M - 1) * np.eye(M) + (inp["Yb"][0].T * inp["rinv_loc"][0]) @ inp["Yb"][0]
    W = out["W"][0]
    assert np.abs(W @ Q @ W - (M - 1) * np.eye(M)).max() <= 1e-13 * (M - 1)


# P-10 ------------------------------------------------------------------------------------
@pytest.mark.parametrize("M,p,scale", [(64, 98, 0.1), (48, 49, 1.0), (32, 3, 1.0)])
def test_evd_free_matrix_function_route(oracle, M, p, scale):
    """A^-1/2 by the Denman-Beavers iteration and A^-1 g by Cholesky, no EVD anywhere."""
    inp = wl.analysis_inputs(batch=2, M=M, p=p, config_index=600 + M, yb_scale=scale)
    out = _run(oracle, inp)
    for b in range(2):
        Yb, r, d = inp["Yb"][b], inp["rinv_loc"][b], inp["d"][b]
        A = (M - 1) / inp["rho"] * np.eye(M) + (Yb.T * r) @ Yb
        # Denman-Beavers: Y -> A^1/2, Z -> A^-1/2 (scaled for fast convergence)
        s = np.linalg.norm(A, 2)
        Y, Z = A / s, np.eye(M)
        for _ in range(60):
            Yn = 0.5 * (Y + gauss_solve(Z, np.eye(M)))
            Zn = 0.5 * (Z + gauss_solve(Y, np.eye(M)))
            done = np.abs(Yn - Y).max() <= 1e-16
            Y, Z = Yn, Zn
            if done:
                break
        W_db = math.sqrt(M - 1) * Z / math.sqrt(s)
        # Cholesky written out
        L = np.zeros((M, M))
        for i in range(M):
            for j in range(i + 1):
                acc = A[i, j] - L[i, :j] @ L[j, :j]
                L[i, j] = math.sqrt(acc) if i == j else acc / L[j, j]
        g = Yb.T @ (r * d)
        z = np.zeros(M)
        for i in range(M):
            z[i] = (g[i] - L[i, :i] @ z[:i]) / L[i, i]
        x = np.zeros(M)
        for i in range(M - 1, -1, -1):
            x[i] = (z[i] - L[i + 1:, i] @ x[i + 1:]) / L[i, i]
        assert np.linalg.norm(out["W"][b] - W_db) <= 1e-12 * np.linalg.norm(W_db)
        assert np.linalg.norm(out["wbar"][b] - x) <= 1e-12 * max(np.linalg.norm(x), 1e-300)


# P-11 ------------------------------------------------------------------------------------
def test_padding_and_permutation_invariance(oracle):
    M, p, ns = 24, 30, 9
    inp = wl.analysis_inputs(batch=2, M=M, p=p, nstate=ns, config_index=81)
    base = _run(oracle, inp)
    rng = np.random.Generator(np.random.Philox(key=5))
    # (a) append zero-weight observations carrying garbage (reading G7)
    pad = 11
    Yb2 = np.concatenate([inp["Yb"], 1e3 * rng.standard_normal((2, pad, M))], axis=1)
    d2 = np.concatenate([inp["d"], 1e3 * rng.standard_normal((2, pad))], axis=1)
    r2 = np.concatenate([inp["rinv_loc"], np.zeros((2, pad))], axis=1)
    out = oracle.letkf_analysis_batched(Yb2, d2, r2, inp["Xb"], inp["rho"])
    assert np.abs(out["W"] - base["W"]).max() <= 1e-14
    assert np.abs(out["Xa"] - base["Xa"]).max() <= 1e-14
    # (b) permute the observations
    perm = rng.permutation(p)
    out = oracle.letkf_analysis_batched(inp["Yb"][:, perm], inp["d"][:, perm],
                                        inp["rinv_loc"][:, perm], inp["Xb"], inp["rho"])
    assert np.abs(out["W"] - base["W"]).max() <= 1e-13
    assert np.abs(out["Xa"] - base["Xa"]).max() <= 1e-13
    # (c) permute the ensemble members
    pm = rng.permutation(M)
    out = oracle.letkf_analysis_batched(inp["Yb"][:, :, pm], inp["d"], inp["rinv_loc"],
                                        inp["Xb"][:, :, pm], inp["rho"])
    assert np.abs(out["W"] - base["W"][:, pm][:, :, pm]).max() <= 1e-13
    assert np.abs(out["Xa"] - base["Xa"][:, :, pm]).max() <= 1e-13


def test_golden_fixture(oracle):
    """Stored values written by tests/golden/make_golden.py (which calls only oracle/)."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "analysis_M6_p4_ns2.txt")
    vals = np.loadtxt(path)
    inp = wl.analysis_inputs(batch=1, M=6, p=4, nstate=2, config_index=9001)
    out = _run(oracle, inp)
    got = np.concatenate([out["Xa"].ravel(), out["wbar"].ravel(), out["W"].ravel()])
    assert np.abs(got - vals).max() <= 1e-14

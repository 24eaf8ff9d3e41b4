"""Tolerance checks shared by the GPU parity tests (north_star):
  (i)   max_k |w_gpu - w_oracle| <= 1e-12 ||A||_2          (||A||_2 = max |w_oracle|)
  (ii)  ||A V - V diag(w)||_F / ||A||_F <= 1e-12
  (iii) max |V^T V - I| <= 1e-12
  (iv)  ||W_gpu - W_orc||_F / ||W_orc||_F <= 1e-10
  (v)   ||Xa_gpu - Xa_orc||_F / ||Xa_orc||_F <= 1e-10, and the same on the increment Xa - xbar 1^T
Pure numpy, evaluated in fp64 on the host.  No arithmetic of the method lives here.
"""
import numpy as np

TOL_W = 1e-12
TOL_RES = 1e-12
TOL_ORTH = 1e-12
TOL_ANALYSIS = 1e-10


def sym_from_lower(A):
    L = np.tril(A)
    return L + np.transpose(np.tril(A, -1), (0, 2, 1))


def evd_errors(A, w, V):
    """Per-matrix (residual, orthogonality) of a claimed EVD; A is the full symmetric input."""
    AV = np.matmul(A, V)
    R = AV - V * w[:, None, :]
    nA = np.sqrt((A * A).sum(axis=(1, 2)))
    nA = np.where(nA > 0, nA, 1.0)
    res = np.sqrt((R * R).sum(axis=(1, 2))) / nA
    G = np.matmul(np.transpose(V, (0, 2, 1)), V)
    G = G - np.eye(V.shape[-1])[None]
    orth = np.abs(G).max(axis=(1, 2))
    return res, orth


def assert_evd(A, w, V, w_ref=None, what=""):
    A = sym_from_lower(A)
    assert np.all(np.isfinite(w)) and np.all(np.isfinite(V)), what
    assert np.all(np.diff(w, axis=1) >= 0), f"{what}: eigenvalues not ascending"
    res, orth = evd_errors(A, w, V)
    assert res.max() <= TOL_RES, f"{what}: residual {res.max():.3e}"
    assert orth.max() <= TOL_ORTH, f"{what}: orthogonality {orth.max():.3e}"
    if w_ref is not None:
        scale = np.abs(w_ref).max(axis=1)
        scale = np.where(scale > 0, scale, 1.0)
        err = (np.abs(w - w_ref).max(axis=1) / scale).max()
        assert err <= TOL_W, f"{what}: eigenvalue error {err:.3e}"
    return res.max(), orth.max()


def rel_fro(x, ref):
    x = x.reshape(x.shape[0], -1)
    ref = ref.reshape(ref.shape[0], -1)
    num = np.sqrt(((x - ref) ** 2).sum(axis=1))
    den = np.sqrt((ref ** 2).sum(axis=1))
    den = np.where(den > 0, den, 1.0)
    return (num / den).max()


def assert_analysis(out, ref, Xb, what=""):
    """out/ref: dicts with Xa (and optionally W, wbar) as numpy arrays."""
    e = rel_fro(out["Xa"], ref["Xa"])
    assert e <= TOL_ANALYSIS, f"{what}: Xa {e:.3e}"
    xbar = Xb.mean(axis=2, keepdims=True)
    e = rel_fro(out["Xa"] - xbar, ref["Xa"] - xbar)
    assert e <= TOL_ANALYSIS, f"{what}: Xa increment {e:.3e}"
    if out.get("W") is not None:
        e = rel_fro(out["W"], ref["W"])
        assert e <= TOL_ANALYSIS, f"{what}: W {e:.3e}"
    if out.get("wbar") is not None:
        # relative to ||wbar_ref||_inf per grid point; where the reference is identically 0 (d = 0,
        # closed form P-9) the product must return (numerically) 0 as well
        num = np.abs(out["wbar"] - ref["wbar"]).reshape(ref["wbar"].shape[0], -1).max(axis=1)
        den = np.abs(ref["wbar"]).reshape(ref["wbar"].shape[0], -1).max(axis=1)
        zero = den == 0.0
        assert (num[zero] <= 1e-14).all(), f"{what}: wbar where the reference is 0: {num[zero].max():.3e}"
        if (~zero).any():
            e = (num[~zero] / den[~zero]).max()
            assert e <= TOL_ANALYSIS, f"{what}: wbar {e:.3e}"

"""GPU parity of letkf_syev_batched_f32 (Table I PAPER.md:189-198:
the paper's precision and sizes).  Reference: the fp64 oracle on the SAME float-rounded inputs.
Tolerances (derived from the arithmetic: fp32 Householder reduction and
back-transform of order M <= 64, fp64 tridiagonal eigenproblem in between):
  max_k |w - w_oracle| <= 50 eps32 ||A||_2,  ||A V - V diag(w)||_F / ||A||_F <= 100 eps32,
  max |V^T V - I| <= 100 eps32,   eps32 = 2^-24."""
import numpy as np
import pytest

from harness import workloads as wl
import parity

pytestmark = pytest.mark.gpu
EPS32 = 2.0 ** -24


@pytest.fixture(scope="module")
def lk():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_2308_03310_b200 import build, letkf
    build.build()
    letkf.load()
    return letkf


def run(lk, A32, **kw):
    import torch
    At = torch.from_numpy(np.ascontiguousarray(A32)).cuda()
    w, V, info = lk.syev_batched_f32(At, **kw)
    torch.cuda.synchronize()
    return w.cpu().numpy().astype(np.float64), V.cpu().numpy().astype(np.float64), info.cpu().numpy()


def check(A32, w, V, wo, what):
    A = parity.sym_from_lower(A32.astype(np.float64))
    assert np.all(np.isfinite(w)) and np.all(np.isfinite(V)), what
    assert np.all(np.diff(w, axis=1) >= 0), f"{what}: eigenvalues not ascending"
    res, orth = parity.evd_errors(A, w, V)
    assert res.max() <= 100 * EPS32, f"{what}: residual {res.max():.3e}"
    assert orth.max() <= 100 * EPS32, f"{what}: orthogonality {orth.max():.3e}"
    scale = np.abs(wo).max(axis=1)
    scale = np.where(scale > 0, scale, 1.0)
    err = (np.abs(w - wo).max(axis=1) / scale).max()
    assert err <= 50 * EPS32, f"{what}: eigenvalue error {err:.3e}"


@pytest.mark.parametrize("M,p", [(16, 49), (32, 49), (48, 49), (64, 98)])
def test_table1_shapes(lk, oracle, M, p):
    """The paper's Table I sizes on LETKF-shaped matrices (configs 2 / 3 / 5), rounded to float."""
    A32 = wl.letkf_shaped(300, M, p, config_index=1200 + M).astype(np.float32)
    w, V, info = run(lk, A32)
    assert (info == 0).all()
    wo, _, _, _ = oracle.syev_batched(A32.astype(np.float64))
    check(A32, w, V, wo, f"f32 M={M}")


@pytest.mark.parametrize("M", [1, 2, 3, 5, 17, 31, 33, 47, 57, 63])
def test_any_order(lk, oracle, M):
    rng = np.random.Generator(np.random.Philox(key=1300 + M))
    G = rng.standard_normal((41, M, M))
    A32 = (G + np.transpose(G, (0, 2, 1))).astype(np.float32)
    w, V, info = run(lk, A32)
    assert (info == 0).all()
    wo, _, _, _ = oracle.syev_batched(A32.astype(np.float64))
    check(A32, w, V, wo, f"f32 random symmetric M={M}")


@pytest.mark.parametrize("p", [0, 3, 48])
def test_paper_shaped_clusters(lk, oracle, p):
    """Dense / sparse observation shapes: (M - p)-fold cluster, zero Householder
    columns, the logging route of the eigensolver."""
    A32 = wl.letkf_shaped(64, 64, p, config_index=1400 + p).astype(np.float32)
    w, V, info = run(lk, A32)
    assert ((info & 0xFFFF) == 0).all()
    wo, _, _, _ = oracle.syev_batched(A32.astype(np.float64))
    check(A32, w, V, wo, f"f32 clusters p={p}")


def test_full_size_and_in_place(lk, oracle):
    """Table I's M = 64 at batch 16384 (the launch configuration bench.py times): validity of every
    matrix, eigenvalues against the oracle on a strided sample; in place; empty batch."""
    import torch
    A32 = wl.config3().astype(np.float32)
    At = torch.from_numpy(A32).cuda()
    w, V, info = lk.syev_batched_f32(At)
    torch.cuda.synchronize()
    assert int(info.abs().max()) == 0
    Ad = At.double()
    Af = torch.tril(Ad) + torch.tril(Ad, -1).transpose(1, 2)
    Vd, wd = V.double(), w.double()
    worst_res = worst_orth = 0.0
    for b0 in range(0, A32.shape[0], 2048):
        sl = slice(b0, b0 + 2048)
        R = torch.matmul(Af[sl], Vd[sl]) - Vd[sl] * wd[sl].unsqueeze(1)
        worst_res = max(worst_res, float((R.flatten(1).norm(dim=1) / Af[sl].flatten(1).norm(dim=1)).max()))
        G = torch.matmul(Vd[sl].transpose(1, 2), Vd[sl]) - torch.eye(64, dtype=torch.float64, device="cuda")
        worst_orth = max(worst_orth, float(G.abs().max()))
    assert worst_res <= 100 * EPS32 and worst_orth <= 100 * EPS32, (worst_res, worst_orth)
    sel = np.arange(0, A32.shape[0], 256)
    wo, _, _, _ = oracle.syev_batched(A32[sel].astype(np.float64))
    wg = w[torch.from_numpy(sel).cuda()].cpu().numpy().astype(np.float64)
    assert (np.abs(wg - wo).max(axis=1) / np.abs(wo).max(axis=1)).max() <= 50 * EPS32
    B = At[:500].clone()
    w2, V2, _ = lk.syev_batched_f32(B, V=B)
    torch.cuda.synchronize()
    assert V2.data_ptr() == B.data_ptr()
    wo2, _, _, _ = oracle.syev_batched(A32[:100].astype(np.float64))
    check(A32[:100], w2[:100].cpu().numpy().astype(np.float64), V2[:100].cpu().numpy().astype(np.float64), wo2, "f32 in place")
    w0, V0, i0 = lk.syev_batched_f32(At[:0])
    assert w0.shape == (0, 64) and V0.shape == (0, 64, 64)
    with pytest.raises(lk.LetkfError):
        lk.syev_batched_f32(torch.zeros((2, 65, 65), dtype=torch.float32, device="cuda"))

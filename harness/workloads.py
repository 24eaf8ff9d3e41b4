"""Seeded synthetic workloads (inputs only) for the LETKF hot path.

This module is the ONE piece shared by the CUDA path's tests/bench and the CPU oracle's
tests: it draws inputs and nothing else.  It contains none of the method's arithmetic
(no EVD, no transform matrix, no ensemble update) and imports neither ``oracle`` nor the
CUDA binding.  The ``syev`` configurations hand the solver a symmetric matrix with the
structure BASELINE.json prescribes; building that *input* needs one matmul, done here with
numpy -- the analysis path's own Gram step (Eq.17) lives separately in oracle/oracle.c and
in csrc/, and neither calls this file to compute its result.

The inputs stand in for the paper's "batched matrix data ... generated from the LBM-LETKF
model", which are not available; shapes and structure follow
BASELINE.json ``configs`` and SURVEY.md section 8(d).  Recipe is restated in DESIGN.md.

RNG: numpy.random.Generator(numpy.random.Philox(key=SEED0 + config_index)); draw order as
written below.  A smaller ``batch`` yields a prefix-compatible stream only per array.
"""
import numpy as np

SEED0 = 230803310
SIGMA_O = 0.1          # observation error std (BASELINE.json configs 2-4)
RHO = 1.1              # multiplicative inflation (BASELINE.json)
LOC_SIGMA = 2.0        # Gaussian localisation length, exp(-d^2 / (2 * 2^2))

SWEEP_M = (16, 32, 48, 64, 96, 128, 192, 256)


def _rng(config_index):
    return np.random.Generator(np.random.Philox(key=SEED0 + config_index))


def patch_weights(ncomp):
    """r_j = l_j / sigma_o^2 over a 7x7 patch, repeated for ``ncomp`` observed components.

    j = c*49 + (dy+3)*7 + (dx+3); l = exp(-(dx^2+dy^2)/(2*LOC_SIGMA^2)).
    """
    off = np.arange(-3, 4, dtype=np.float64)
    dy, dx = np.meshgrid(off, off, indexing="ij")
    ell = np.exp(-(dx * dx + dy * dy) / (2.0 * LOC_SIGMA * LOC_SIGMA)).reshape(-1)
    return np.tile(ell / (SIGMA_O * SIGMA_O), ncomp)


def weights_for_p(p):
    """Localisation-weighted inverse obs variance for an arbitrary p (truncated/tiled patch)."""
    if p == 0:
        return np.zeros(0)
    ncomp = (p + 48) // 49
    return patch_weights(ncomp)[:p].copy()


def known_spectrum(batch=1024, M=32, config_index=1, nreflect=None):
    """Config 1: A_b = Q_b diag(lam_b) Q_b^T, lam ~ U[1,100], Q_b = product of M reflectors.

    Returns (A[batch][M][M], lam_sorted[batch][M]).
    """
    rng = _rng(config_index)
    nreflect = M if nreflect is None else nreflect
    lam = rng.uniform(1.0, 100.0, size=(batch, M))
    v = rng.standard_normal(size=(batch, nreflect, M))
    A = np.zeros((batch, M, M))
    idx = np.arange(M)
    A[:, idx, idx] = lam
    for i in range(nreflect):
        u = v[:, i, :]
        beta = 2.0 / np.einsum("bm,bm->b", u, u)
        # A <- H A H,  H = I - beta u u^T  (applied as two rank-1 corrections)
        Au = np.einsum("bmn,bn->bm", A, u)
        A -= beta[:, None, None] * Au[:, :, None] * u[:, None, :]
        uA = np.einsum("bm,bmn->bn", u, A)
        A -= beta[:, None, None] * u[:, :, None] * uA[:, None, :]
    A = 0.5 * (A + np.transpose(A, (0, 2, 1)))
    return A, np.sort(lam, axis=1)


def centred_normal(rng, batch, p, M, scale=1.0):
    """Yb[batch][p][M] ~ N(0, scale^2), each row centred across the ensemble (Eq.19)."""
    Yb = rng.standard_normal(size=(batch, p, M))
    if scale != 1.0:
        Yb *= scale
    if M > 0 and p > 0:
        Yb -= Yb.mean(axis=2, keepdims=True)
    return Yb


def letkf_shaped(batch, M, p, config_index, rho=RHO, chunk=2048):
    """Configs 2, 3, 5: A_b = ((M-1)/rho) I + Yb^T diag(r) Yb with Yb ~ N(0,1) row-centred.

    Returns A[batch][M][M] (symmetric by construction).
    """
    rng = _rng(config_index)
    r = weights_for_p(p)
    A = np.empty((batch, M, M))
    idx = np.arange(M)
    for b0 in range(0, batch, chunk):
        b1 = min(batch, b0 + chunk)
        Yb = centred_normal(rng, b1 - b0, p, M)
        if p > 0:
            G = np.matmul(np.transpose(Yb, (0, 2, 1)) * r[None, None, :], Yb)
            G = 0.5 * (G + np.transpose(G, (0, 2, 1)))
        else:
            G = np.zeros((b1 - b0, M, M))
        G[:, idx, idx] += (M - 1) / rho
        A[b0:b1] = G
    return A


def config2(batch=16384):
    return letkf_shaped(batch, 48, 49, 2)


def config3(batch=16384):
    return letkf_shaped(batch, 64, 98, 3)


def sweep_batch(M):
    """Config 5 batch: batch * M^2 ~ 64 Mi elements."""
    return (1 << 26) // (M * M)


def sweep_p(M):
    """Config 5 reading G17: p = 49 for M <= 48, 98 from M = 64 up."""
    return 49 if M <= 48 else 98


def config5(M, batch=None):
    batch = sweep_batch(M) if batch is None else batch
    return letkf_shaped(batch, M, sweep_p(M), 50 + SWEEP_M.index(M) if M in SWEEP_M else 5)


def analysis_inputs(batch=16384, M=64, p=98, nstate=9, config_index=4,
                    zero_weight_fraction=0.0, yb_scale=0.1):
    """Config 4 (and the paper-shaped extras with other p).

    Xb[batch][nstate][M] ~ N(1/9, 0.01^2); Yb[batch][p][M] ~ N(0, 0.1^2) row-centred;
    d[batch][p] ~ N(0, 0.1^2); rinv_loc[batch][p] = patch weights replicated per point,
    optionally with a random fraction set to zero (padded observations, reading G7).
    """
    rng = _rng(config_index)
    Xb = 1.0 / 9.0 + 0.01 * rng.standard_normal(size=(batch, nstate, M))
    Yb = centred_normal(rng, batch, p, M, scale=yb_scale)
    d = 0.1 * rng.standard_normal(size=(batch, p))
    rinv = np.broadcast_to(weights_for_p(p), (batch, p)).copy()
    if zero_weight_fraction > 0.0 and p > 0:
        mask = rng.uniform(size=(batch, p)) < zero_weight_fraction
        rinv[mask] = 0.0
    return dict(Yb=Yb, d=d, rinv_loc=rinv, Xb=Xb, rho=RHO, M=M, p=p, nstate=nstate)


def toeplitz_tridiagonal(M, a=0.0, b=1.0):
    """tridiag(b, a, b) of order M: eigenvalues a + 2 b cos(k pi / (M+1))."""
    A = np.zeros((M, M))
    i = np.arange(M)
    A[i, i] = a
    A[i[:-1], i[:-1] + 1] = b
    A[i[:-1] + 1, i[:-1]] = b
    return A


def grid_inputs(Ny=128, Nx=128, M=64, V=2, nstate=9, config_index=6, obs_every=1):
    """Grid form of config 4: instead of a materialised Y_loc the
    forecast observations of the whole periodic grid, Yf[V][Ny][Nx][M] ~ 0.05 + N(0, 0.1^2) (NOT
    centred: Eq.18-19 are part of the path), observations yo[V][Ny][Nx] ~ 0.05 + N(0, 0.1^2),
    background ensemble Xb[Ny*Nx][nstate][M] ~ N(1/9, 0.01^2) and a mask of observed points (every
    `obs_every`-th point in x and y, "spacing of observation points"; 1 = all)."""
    rng = _rng(config_index)
    Yf = 0.05 + 0.1 * rng.standard_normal(size=(V, Ny, Nx, M))
    yo = 0.05 + 0.1 * rng.standard_normal(size=(V, Ny, Nx))
    Xb = 1.0 / 9.0 + 0.01 * rng.standard_normal(size=(Ny * Nx, nstate, M))
    mask = np.zeros((Ny, Nx), dtype=np.uint8)
    mask[::obs_every, ::obs_every] = 1
    return dict(Yf=Yf, yo=yo, Xb=Xb, mask=mask, rho=RHO, sigma_o=SIGMA_O, hw=3, loc_kind=0, L=2.0)

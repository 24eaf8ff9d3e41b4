"""Pins of the grid form of the oracle (local-observation gather,
Eq.18-19 and the localisation function fused in front of the local analysis; PAPER.md:144-151,
Procedure 1 lines 1-2).  CPU only."""
import numpy as np
import pytest

from harness import workloads as wl


def gather_numpy(Yf, yo, mask, hw, weight):
    """Y_loc materialised with numpy.roll (independent of the oracle's index arithmetic):
    returns Yb[Ny*Nx][p][M] (centred), d[Ny*Nx][p], r[Ny*Nx][p] (without 1/sigma^2)."""
    V, Ny, Nx, M = Yf.shape
    ybar = Yf.mean(axis=3)
    rows, dd, rr = [], [], []
    for v in range(V):
        for dy in range(-hw, hw + 1):
            for dx in range(-hw, hw + 1):
                Ys = np.roll(Yf[v], shift=(-dy, -dx), axis=(0, 1))          # [y][x] <- [y+dy][x+dx]
                bs = np.roll(ybar[v], shift=(-dy, -dx), axis=(0, 1))
                os_ = np.roll(yo[v], shift=(-dy, -dx), axis=(0, 1))
                ms = np.roll(mask, shift=(-dy, -dx), axis=(0, 1))
                rows.append((Ys - bs[..., None]).reshape(Ny * Nx, M))
                dd.append((os_ - bs).reshape(Ny * Nx))
                rr.append((weight(np.hypot(dx, dy)) * (ms != 0)).reshape(Ny * Nx))
    return np.stack(rows, axis=1), np.stack(dd, axis=1), np.stack(rr, axis=1)


@pytest.mark.parametrize("loc_kind,L,obs_every", [(0, 2.0, 1), (1, 2.0, 1), (1, 1.5, 2), (0, 1.0, 3)])
def test_grid_equals_batched_on_gathered_inputs(oracle, loc_kind, L, obs_every):
    g = wl.grid_inputs(Ny=6, Nx=9, M=8, V=2, nstate=3, config_index=61, obs_every=obs_every)
    hw, sig = 2, g["sigma_o"]
    w = np.vectorize(lambda dist: oracle.localisation(loc_kind, L, dist))
    Yb, d, r = gather_numpy(g["Yf"], g["yo"], g["mask"], hw, w)
    ref = oracle.letkf_analysis_batched(Yb, d, r / sig ** 2, g["Xb"], g["rho"])
    got = oracle.letkf_analysis_grid(g["Yf"], g["yo"], g["Xb"], hw, loc_kind, L, sig, g["rho"], mask=g["mask"])
    assert (got["info"] == 0).all()
    assert np.abs(got["Xa"] - ref["Xa"]).max() <= 1e-13
    assert np.abs(got["wbar"] - ref["wbar"]).max() <= 1e-12 * max(1.0, np.abs(ref["wbar"]).max())


def test_grid_is_translation_equivariant(oracle):
    """Periodic domain: shifting every field by (sy, sx) shifts the analysis the same way."""
    g = wl.grid_inputs(Ny=5, Nx=7, M=6, V=1, nstate=2, config_index=62)
    a = oracle.letkf_analysis_grid(g["Yf"], g["yo"], g["Xb"], 1, 1, 1.2, 0.1, 1.1)
    sy, sx = 2, 3
    Yf2 = np.roll(g["Yf"], (sy, sx), axis=(1, 2))
    yo2 = np.roll(g["yo"], (sy, sx), axis=(1, 2))
    Xb2 = np.roll(g["Xb"].reshape(5, 7, 2, 6), (sy, sx), axis=(0, 1)).reshape(35, 2, 6)
    b = oracle.letkf_analysis_grid(Yf2, yo2, Xb2, 1, 1, 1.2, 0.1, 1.1)
    Xa_shift = np.roll(a["Xa"].reshape(5, 7, 2, 6), (sy, sx), axis=(0, 1)).reshape(35, 2, 6)
    assert np.abs(b["Xa"] - Xa_shift).max() <= 1e-13


def test_unobserved_grid_changes_nothing_but_inflation(oracle):
    """mask == 0 everywhere: no observations, Xa = xbar + sqrt(rho) dX (closed form P-9)."""
    g = wl.grid_inputs(Ny=4, Nx=4, M=5, V=2, nstate=2, config_index=63)
    out = oracle.letkf_analysis_grid(g["Yf"], g["yo"], g["Xb"], 1, 0, 2.0, 0.1, 1.21, mask=np.zeros((4, 4)))
    xbar = g["Xb"].mean(axis=2, keepdims=True)
    assert np.abs(out["Xa"] - (xbar + 1.1 * (g["Xb"] - xbar))).max() <= 1e-13
    assert np.abs(out["wbar"]).max() <= 1e-14


def test_gaspari_cohn_is_the_tent_self_convolution(oracle):
    """The 5th-order piecewise rational of ref.[21] is the self-convolution over R^3 of the tent
    (1 - r/c)_+, normalised at 0: checked by brute-force quadrature of that definition,
    (h*h)(d) = (2 pi / d) int_0^c h(r) r int_{|d-r|}^{min(d+r,c)} h(s) s ds dr."""
    c = 1.7

    def tent(r):
        return np.clip(1.0 - r / c, 0.0, None)

    def conv(dist, n=1500):
        r = (np.arange(n) + 0.5) * (c / n)
        tot = 0.0
        for ri in r:
            lo, hi = abs(dist - ri), min(dist + ri, c)
            if hi > lo:
                s = lo + (np.arange(300) + 0.5) * ((hi - lo) / 300)
                tot += tent(ri) * ri * np.sum(tent(s) * s) * ((hi - lo) / 300) * (c / n)
        return 2.0 * np.pi / dist * tot

    c0 = conv(1e-3 * c)
    for z in (0.3, 0.8, 1.0, 1.4, 1.95):
        assert abs(conv(z * c) / c0 - oracle.localisation(1, c, z * c)) <= 2e-5
    assert oracle.localisation(1, c, 0.0) == 1.0
    assert oracle.localisation(1, c, 2.0 * c) == 0.0 and oracle.localisation(1, c, 5.0 * c) == 0.0
    assert abs(oracle.localisation(1, c, c) - 5.0 / 24.0) <= 1e-15
    zs = np.linspace(0.0, 2.0, 401) * c
    vals = np.array([oracle.localisation(1, c, z) for z in zs])
    assert (np.diff(vals) <= 1e-16).all() and (vals >= 0).all()              # monotone, non-negative
    assert abs(oracle.localisation(0, 2.0, 2.0) - np.exp(-0.5)) <= 1e-16    # Gaussian of BASELINE.json

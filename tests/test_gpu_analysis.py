"""GPU parity: letkf_analysis_batched (through the C ABI) against the CPU oracle.
PAPER.md:120-146 (Eq.13-19); tolerances of north_star / parity.py."""
import math

import numpy as np
import pytest

from harness import workloads as wl
import parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lk():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_2308_03310_b200 import build, letkf
    build.build()
    letkf.load()
    return letkf


def run_gpu(lk, inp, want_W=True, want_wbar=True, rho=None, **kw):
    import torch
    t = {k: torch.from_numpy(np.ascontiguousarray(inp[k])).cuda() for k in ("Yb", "d", "rinv_loc", "Xb")}
    out = lk.analysis_batched(t["Yb"], t["d"], t["rinv_loc"], t["Xb"], inp["rho"] if rho is None else rho,
                              want_W=want_W, want_wbar=want_wbar, **kw)
    torch.cuda.synchronize()
    return {k: (v.cpu().numpy() if v is not None else None) for k, v in out.items()}


def run_oracle(oracle, inp, rho=None):
    return oracle.letkf_analysis_batched(inp["Yb"], inp["d"], inp["rinv_loc"], inp["Xb"],
                                         inp["rho"] if rho is None else rho)


@pytest.mark.parametrize("M,p,ns,batch", [(64, 98, 9, 200), (64, 3, 9, 65), (64, 48, 9, 64), (48, 49, 9, 100),
                                          (32, 49, 9, 100), (16, 5, 3, 77), (6, 4, 2, 5), (2, 7, 1, 9),
                                          (33, 20, 4, 21), (96, 98, 9, 6), (130, 98, 9, 3)])
def test_analysis_vs_oracle(lk, oracle, M, p, ns, batch):
    """BASELINE config 4 shape (reduced batch), the paper's dense (p=3) and sparse (p=48) shapes,
    and ragged / odd sizes."""
    inp = wl.analysis_inputs(batch=batch, M=M, p=p, nstate=ns, config_index=400 + M + p)
    out = run_gpu(lk, inp)
    ref = run_oracle(oracle, inp)
    assert (out["info"] == 0).all()
    parity.assert_analysis(out, ref, inp["Xb"], f"M={M} p={p} ns={ns}")


@pytest.mark.gpu
@pytest.mark.parametrize("M,p,ns,batch", [(70, 5, 3, 4), (96, 0, 2, 3), (97, 1, 1, 2), (128, 230, 4, 2), (256, 130, 17, 2)])
def test_analysis_above_64_gram_shapes(lk, oracle, M, p, ns, batch):
    """The Gram kernel of the orders above 64 (big_gram, FP64 tensor cores): a number of observations that is not a
    multiple of four, none at all, one, more than one shared-memory chunk holds (M = 128: 212; M = 256: 108), ragged
    orders; nstate above eight (two rounds of the epilogue's grouped reductions)."""
    inp = wl.analysis_inputs(batch=batch, M=M, p=p, nstate=ns, config_index=900 + M + p)
    out = run_gpu(lk, inp, want_wbar=True)
    ref = run_oracle(oracle, inp)
    assert (out["info"] == 0).all()
    parity.assert_analysis(out, ref, inp["Xb"], f"M={M} p={p} ns={ns}")


@pytest.mark.parametrize("want_W", [True, False])
@pytest.mark.parametrize("M,batch", [(128, 4), (160, 3), (192, 3), (256, 2)])
def test_analysis_large_ensembles(lk, oracle, M, batch, want_W):
    """LETKF_MAX_M = 256 applies to the analysis call as well: the paths above the register kernels
    (shared-memory resident up to 160, any-M kernels beyond), with the transform matrix requested
    and not."""
    inp = wl.analysis_inputs(batch=batch, M=M, p=98, nstate=9, config_index=430 + M)
    out = run_gpu(lk, inp, want_W=want_W, want_wbar=True)
    ref = run_oracle(oracle, inp)
    assert (out["info"] == 0).all()
    assert (out["W"] is not None) == want_W
    parity.assert_analysis(out, ref, inp["Xb"], f"M={M} W={want_W}")


@pytest.mark.parametrize("opt", ["qform", "evec"])
@pytest.mark.parametrize("M,p,ns", [(64, 98, 9), (48, 49, 9), (20, 7, 3), (64, 98, 15)])
def test_fused_analysis_other_forms(lk, oracle, M, p, ns, opt):
    """The fused epilogue behind the other forms of the apply kernel: explicit Q (qform = 1) and
    replayed rotations only (evec = 0); the default is covered by test_fused_epilogue_vs_oracle."""
    inp = wl.analysis_inputs(batch=70, M=M, p=p, nstate=ns, config_index=450 + M)
    try:
        lk.set_option(opt, 1 if opt == "qform" else 0)
        out = run_gpu(lk, inp, want_W=False, want_wbar=True)
    finally:
        lk.set_option("qform", 0)
        lk.set_option("evec", 1)
    ref = run_oracle(oracle, inp)
    assert (out["info"] == 0).all()
    parity.assert_analysis(out, ref, inp["Xb"], f"{opt} M={M}")


def test_without_optional_outputs_and_in_place(lk, oracle):
    import torch
    inp = wl.analysis_inputs(batch=50, M=64, p=98, nstate=9, config_index=41)
    ref = run_oracle(oracle, inp)
    out = run_gpu(lk, inp, want_W=False, want_wbar=False)
    assert out["W"] is None and out["wbar"] is None
    parity.assert_analysis(out, ref, inp["Xb"], "no W")
    t = {k: torch.from_numpy(inp[k]).cuda() for k in ("Yb", "d", "rinv_loc", "Xb")}
    Xb = t["Xb"].clone()
    o2 = lk.analysis_batched(t["Yb"], t["d"], t["rinv_loc"], Xb, inp["rho"], Xa=Xb)
    torch.cuda.synchronize()
    assert o2["Xa"].data_ptr() == Xb.data_ptr()
    parity.assert_analysis({"Xa": Xb.cpu().numpy()}, ref, inp["Xb"], "in place")


def test_no_observations_closed_form(lk):
    """p = 0 (pin P-9): A = ((M-1)/rho) I, W = sqrt(rho) I, wbar = 0, Xa = xbar + sqrt(rho) dX."""
    inp = wl.analysis_inputs(batch=7, M=64, p=0, nstate=9, config_index=42)
    out = run_gpu(lk, inp)
    xbar = inp["Xb"].mean(axis=2, keepdims=True)
    exact = xbar + math.sqrt(inp["rho"]) * (inp["Xb"] - xbar)
    assert np.abs(out["Xa"] - exact).max() <= 1e-13
    assert np.abs(out["W"] - math.sqrt(inp["rho"]) * np.eye(64)).max() <= 1e-13
    assert np.abs(out["wbar"]).max() == 0.0


def test_zero_weights_are_padding(lk, oracle):
    """Reading G7 (PAPER.md:151 l_max padding): zero-weight observations do not matter."""
    inp = wl.analysis_inputs(batch=30, M=64, p=98, nstate=9, config_index=43, zero_weight_fraction=0.25)
    out = run_gpu(lk, inp)
    ref = run_oracle(oracle, inp)
    parity.assert_analysis(out, ref, inp["Xb"], "25% zero weights")
    junk = dict(inp)
    junk["Yb"] = inp["Yb"].copy()
    junk["d"] = inp["d"].copy()
    mask = inp["rinv_loc"] == 0.0
    junk["Yb"][mask] = 123.0
    junk["d"][mask] = -7.0
    out2 = run_gpu(lk, junk)
    assert parity.rel_fro(out2["Xa"], out["Xa"]) <= 1e-13


def test_rho_one_is_eq17(lk, oracle):
    inp = wl.analysis_inputs(batch=20, M=64, p=98, nstate=9, config_index=44)
    out = run_gpu(lk, inp, rho=1.0)
    ref = run_oracle(oracle, inp, rho=1.0)
    parity.assert_analysis(out, ref, inp["Xb"], "rho=1")


def test_structural_identities_full_size(lk, oracle):
    """BASELINE config 4 at full size (128x128 points, the launch configuration bench.py times):
    pins P-8 on every point -- W symmetric, W 1 = sqrt(rho) 1, mean(Xa) = xbar + dX wbar --
    plus oracle parity on a strided sample."""
    import torch
    inp = wl.analysis_inputs()                       # batch=16384, M=64, p=98, ns=9
    t = {k: torch.from_numpy(inp[k]).cuda() for k in ("Yb", "d", "rinv_loc", "Xb")}
    out = lk.analysis_batched(t["Yb"], t["d"], t["rinv_loc"], t["Xb"], inp["rho"], want_W=True, want_wbar=True)
    torch.cuda.synchronize()
    assert int(out["info"].abs().max()) == 0
    W, wbar, Xa, Xb = out["W"], out["wbar"], out["Xa"], t["Xb"]
    assert float((W - W.transpose(1, 2)).abs().max()) <= 1e-12
    assert float((W.sum(dim=2) - math.sqrt(inp["rho"])).abs().max()) <= 1e-11
    xbar = Xb.mean(dim=2, keepdim=True)
    dX = Xb - xbar
    mean_pred = xbar.squeeze(2) + torch.einsum("bsm,bm->bs", dX, wbar) \
        + (math.sqrt(inp["rho"]) - 1.0) * 0.0
    # mean over members of dX W = dX (W 1)/M = sqrt(rho) dX 1 / M = 0
    assert float((Xa.mean(dim=2) - mean_pred).abs().max()) <= 1e-12
    sel = np.arange(0, 16384, 256)
    sub = {k: (v[sel] if isinstance(v, np.ndarray) else v) for k, v in inp.items()}
    ref = run_oracle(oracle, sub)
    got = {"Xa": Xa.cpu().numpy()[sel], "W": W.cpu().numpy()[sel], "wbar": wbar.cpu().numpy()[sel]}
    parity.assert_analysis(got, ref, sub["Xb"], "config4 sample")
    out2 = lk.analysis_batched(t["Yb"], t["d"], t["rinv_loc"], t["Xb"], inp["rho"])
    torch.cuda.synchronize()
    assert float((out2["Xa"] - Xa).abs().max()) <= 1e-13


def test_host_entry_point_equals_device_call(lk):
    import torch
    inp = wl.analysis_inputs(batch=2048 + 77, M=64, p=98, nstate=9)
    t = {k: torch.from_numpy(inp[k]) for k in ("Yb", "d", "rinv_loc", "Xb")}
    dev = lk.analysis_batched(t["Yb"].cuda(), t["d"].cuda(), t["rinv_loc"].cuda(), t["Xb"].cuda(),
                              inp["rho"], want_W=True, want_wbar=True)
    torch.cuda.synchronize()
    host = lk.analysis_batched_host(t["Yb"].pin_memory(), t["d"].pin_memory(), t["rinv_loc"].pin_memory(),
                                    t["Xb"].pin_memory(), inp["rho"], want_W=True, want_wbar=True)
    for k in ("Xa", "W", "wbar", "info"):
        assert torch.equal(host[k], dev[k].cpu()), k
    # without W the epilogue is fused into the apply kernel (another summation order): bitwise
    # equal to the device call of the same form, and within tolerance of the W form
    lean = lk.analysis_batched_host(t["Yb"], t["d"], t["rinv_loc"], t["Xb"], inp["rho"])   # pageable, no W
    dev_lean = lk.analysis_batched(t["Yb"].cuda(), t["d"].cuda(), t["rinv_loc"].cuda(), t["Xb"].cuda(), inp["rho"])
    torch.cuda.synchronize()
    assert lean["W"] is None and torch.equal(lean["Xa"], dev_lean["Xa"].cpu())
    num = (lean["Xa"] - host["Xa"]).flatten(1).norm(dim=1)
    den = (host["Xa"] - t["Xb"].mean(dim=2, keepdim=True)).flatten(1).norm(dim=1)
    assert float((num / den).max()) <= parity.TOL_ANALYSIS


@pytest.mark.parametrize("M,p,ns,batch", [(64, 98, 9, 200), (64, 3, 9, 65), (64, 48, 9, 64), (64, 0, 9, 8),
                                          (48, 49, 9, 100), (47, 49, 5, 33), (32, 49, 9, 100), (33, 20, 4, 21),
                                          (16, 5, 3, 77), (17, 5, 15, 9), (6, 4, 2, 5), (2, 7, 1, 9),
                                          (64, 98, 16, 7)])
def test_fused_epilogue_vs_oracle(lk, oracle, M, p, ns, batch):
    """Without W the steps a6-a9 run inside the apply kernel on the V held in registers
    (nstate <= 15; nstate = 16 falls back to the any-M epilogue): same tolerances vs the oracle,
    wbar included, and the same answer as the unfused form to rounding."""
    inp = wl.analysis_inputs(batch=batch, M=M, p=p, nstate=ns, config_index=500 + M + p)
    ref = run_oracle(oracle, inp)
    out = run_gpu(lk, inp, want_W=False, want_wbar=True)
    assert (out["info"] == 0).all() and out["W"] is None
    parity.assert_analysis(out, ref, inp["Xb"], f"fused M={M} p={p} ns={ns}")
    full = run_gpu(lk, inp, want_W=True, want_wbar=True)
    parity.assert_analysis(out, full, inp["Xb"], f"fused vs unfused M={M} p={p} ns={ns}")


@pytest.mark.parametrize("opts", [{"evec": 0}, {"qform": 1}])
def test_fused_analysis_on_the_slow_path(lk, oracle, opts):
    """A rotation log too short for the matrix inside the fused analysis: fast_apply<epilogue> runs the
    classic iteration for those points itself (LETKF_INFO_SLOWPATH) and carries on with a6-a9."""
    inp = wl.analysis_inputs(batch=150, M=64, p=98, nstate=9, config_index=45)
    ref = run_oracle(oracle, inp)
    try:
        for k, v in opts.items():
            lk.set_option(k, v)
        lk.set_option("log_shrink", 3)
        out = run_gpu(lk, inp, want_W=False, want_wbar=True)
    finally:
        for k, v in (("log_shrink", 1), ("evec", 1), ("qform", 0)):
            lk.set_option(k, v)
    assert ((out["info"] & 0xFFFF) == 0).all() and (out["info"] & lk.INFO_SLOWPATH).astype(bool).all()
    parity.assert_analysis(out, ref, inp["Xb"], "fused analysis, slow path")


@pytest.mark.parametrize("M,p,ns,batch,scale", [(64, 98, 9, 120, 0.1), (64, 3, 9, 40, 0.1), (64, 48, 9, 40, 0.1),
                                                (48, 49, 9, 50, 0.1), (33, 20, 4, 21, 0.1), (16, 5, 3, 30, 0.1),
                                                (2, 7, 1, 9, 0.1), (64, 98, 9, 30, 1.0), (64, 98, 16, 20, 3.0)])
def test_evdfree_analysis_vs_oracle(lk, oracle, M, p, ns, batch, scale):
    """letkf_analysis_batched_evdfree: W = sqrt(M-1) Q^-1/2 and wbar = Q^-1 g by a
    coupled Newton-Schulz iteration on the FP64 tensor cores, no EVD anywhere -- against the same
    oracle; the 1e-10 tolerances at kappa(Q) ~ 4 (config 4 shape, the paper's p = 3 / 48 shapes, ragged
    sizes), the documented ~3e-14 kappa^2 at kappa ~ 300 (yb_scale 1: config 3's conditioning) and ~ 3e3."""
    import torch
    inp = wl.analysis_inputs(batch=batch, M=M, p=p, nstate=ns, config_index=470 + M + p, yb_scale=scale)
    t = {k: torch.from_numpy(inp[k]).cuda() for k in ("Yb", "d", "rinv_loc", "Xb")}
    out = lk.analysis_batched_evdfree(t["Yb"], t["d"], t["rinv_loc"], t["Xb"], inp["rho"], want_W=True, want_wbar=True)
    torch.cuda.synchronize()
    out = {k: (v.cpu().numpy() if v is not None else None) for k, v in out.items()}
    ref = run_oracle(oracle, inp)
    assert ((out["info"] & lk.INFO_NS_NOCONV) == 0).all() and (out["info"] > 0).all() and (out["info"] <= 24).all()
    if scale <= 0.1:
        parity.assert_analysis(out, ref, inp["Xb"], f"evd-free M={M} p={p} scale={scale}")
    else:
        # kappa(Q) ~ 300 / 3e3: the documented accuracy of the coupled iteration, ~3e-14 kappa^2 (letkf.h)
        xbar = inp["Xb"].mean(axis=2, keepdims=True)
        bound = 3e-9 if scale == 1.0 else 1e-6
        assert parity.rel_fro(out["Xa"] - xbar, ref["Xa"] - xbar) <= bound
        assert parity.rel_fro(out["W"], ref["W"]) <= bound


def test_evdfree_full_size_sample(lk, oracle):
    """Config 4 at full size through the EVD-free form: identities on every grid point (W symmetric,
    W A W = (M-1) I through W 1 = sqrt(rho) 1 and mean preservation), the oracle on a strided sample."""
    import torch
    inp = wl.analysis_inputs()
    t = {k: torch.from_numpy(inp[k]).cuda() for k in ("Yb", "d", "rinv_loc", "Xb")}
    out = lk.analysis_batched_evdfree(t["Yb"], t["d"], t["rinv_loc"], t["Xb"], inp["rho"], want_W=True, want_wbar=True)
    torch.cuda.synchronize()
    assert int((out["info"] & lk.INFO_NS_NOCONV).max()) == 0
    W = out["W"]
    assert float((W - W.transpose(1, 2)).abs().max()) <= 1e-12
    assert float((W.sum(dim=2) - math.sqrt(inp["rho"])).abs().max()) <= 1e-11          # W 1 = sqrt(rho) 1 (P-8)
    sel = np.arange(0, inp["Xb"].shape[0], 512)
    sub = {k: (v[sel] if isinstance(v, np.ndarray) else v) for k, v in inp.items()}
    ref = run_oracle(oracle, sub)
    idx = torch.from_numpy(sel).cuda()
    got = {"Xa": out["Xa"][idx].cpu().numpy(), "W": W[idx].cpu().numpy(), "wbar": out["wbar"][idx].cpu().numpy()}
    parity.assert_analysis(got, ref, sub["Xb"], "evd-free config 4 sample")

"""Small driver for compute-sanitizer (memcheck / racecheck / synccheck): every
kernel family of the library on small batches, sub-chunk pipeline on.  Not collected by pytest.

    compute-sanitizer --tool racecheck python tests/sanitize_run.py [quick]

Exits non-zero if a result is invalid (the sanitizer's own findings are in its report)."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))
from harness import workloads as wl                      # noqa: E402
from paper_2308_03310_b200 import build, letkf           # noqa: E402
import parity                                             # noqa: E402


def main():
    quick = len(sys.argv) > 1 and sys.argv[1] == "quick"
    build.build()
    letkf.load()
    letkf.set_option("sub_chunk", 16)                     # several sub-chunks and slot reuse on tiny batches
    letkf.set_option("slots", 3)
    letkf.set_option("log_slots", 2)
    ran = []
    for M, p in ((48, 49), (64, 98), (64, 48), (96, 98), (128, 98), (192, 98)):
        if quick and M > 64:
            continue
        batch = 40 if M <= 64 else 6
        A = wl.letkf_shaped(batch, M, p, config_index=1500 + M + p)
        for opts in ({"bisect": 0}, {"bisect": 1}, {"evec": 0, "two_pass": 1}, {"qform": 1, "two_pass": 0}):
            if M > 64 and "bisect" in opts and opts["bisect"] == 1:
                continue
            for k, v in opts.items():
                letkf.set_option(k, v)
            w, V, info = letkf.syev_batched(torch.from_numpy(A).cuda())
            torch.cuda.synchronize()
            for k, v in (("bisect", -1), ("evec", 1), ("two_pass", -1), ("qform", 0)):
                letkf.set_option(k, v)
            assert int((info & 0xFFFF).abs().max()) == 0
            parity.assert_evd(A, w.cpu().numpy(), V.cpu().numpy(), None, f"sanitize syev M={M} {opts}")
            ran.append(f"syev M={M} p={p} {opts}")
    A32 = wl.letkf_shaped(40, 64, 98, config_index=1600).astype(np.float32)
    w, V, info = letkf.syev_batched_f32(torch.from_numpy(A32).cuda())
    torch.cuda.synchronize()
    assert int(info.abs().max()) == 0
    ran.append("syev_f32 M=64")
    for M, want_W in ((64, False), (64, True), (48, False), (96, False)):
        if quick and M > 64:
            continue
        inp = wl.analysis_inputs(batch=40 if M <= 64 else 6, M=M, p=98 if M >= 64 else 49, nstate=9, config_index=1700 + M)
        t = {k: torch.from_numpy(inp[k]).cuda() for k in ("Yb", "d", "rinv_loc", "Xb")}
        out = letkf.analysis_batched(t["Yb"], t["d"], t["rinv_loc"], t["Xb"], inp["rho"], want_W=want_W, want_wbar=True)
        torch.cuda.synchronize()
        assert torch.isfinite(out["Xa"]).all() and int(out["info"].abs().max()) == 0
        ran.append(f"analysis M={M} W={want_W}")
    g = wl.grid_inputs(Ny=6, Nx=7, M=64, V=2, nstate=9, config_index=1800, obs_every=2)
    go = letkf.analysis_grid(torch.from_numpy(g["Yf"]).cuda(), torch.from_numpy(g["yo"]).cuda(), torch.from_numpy(g["Xb"]).cuda(),
                             3, 1, 2.0, g["sigma_o"], g["rho"], obs_mask=torch.from_numpy(g["mask"]).cuda())
    torch.cuda.synchronize()
    assert torch.isfinite(go["Xa"]).all()
    ran.append("analysis_grid 6x7 M=64")
    print("sanitize_run ok:", len(ran), "cases")
    for r in ran:
        print("  ", r)


if __name__ == "__main__":
    main()

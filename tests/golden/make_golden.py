"""Writes the stored expected values under tests/golden/.  Calls ONLY oracle/ (and the seeded
input generator); never the CUDA path.  Re-run from the repo root:

    python tests/golden/make_golden.py

analysis_M6_p4_ns2.txt: Xa (2x6), wbar (6), W (6x6) of one grid point, M=6, p=4, nstate=2,
rho=1.1, inputs workloads.analysis_inputs(config_index=9001) -- a regression fixture for the
local analysis Eq.13-17; the values themselves are pinned by the
mathematical tests in tests/test_oracle_letkf.py, not by this file.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from harness import workloads as wl  # noqa: E402


def main():
    inp = wl.analysis_inputs(batch=1, M=6, p=4, nstate=2, config_index=9001)
    out = oracle.letkf_analysis_batched(inp["Yb"], inp["d"], inp["rinv_loc"], inp["Xb"], inp["rho"])
    vals = np.concatenate([out["Xa"].ravel(), out["wbar"].ravel(), out["W"].ravel()])
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "analysis_M6_p4_ns2.txt")
    np.savetxt(path, vals, fmt="%.17e",
               header="oracle.letkf_analysis_batched, M=6 p=4 nstate=2 rho=1.1, "
                      "workloads.analysis_inputs(config_index=9001): Xa(12) wbar(6) W(36)")
    print("wrote", path)


if __name__ == "__main__":
    main()

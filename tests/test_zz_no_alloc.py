"""GPU: letkf_syev_batched_static -- the entry point that allocates nothing (scratch memory in a
file-scope `static __device__` array of the library, letkf.h) -- against letkf_syev_batched, the
existing path, on the same seeded inputs, on calls in a row that share the array.  Tolerances of
parity.py.  (This file sorts last on purpose: the array is shared state of the process.)"""
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


def clustered(batch, M, seed):
    """Spectra with a tight cluster (the matrices that take the logged-rotation route)."""
    rng = np.random.Generator(np.random.Philox(key=seed))
    lam = np.sort(rng.uniform(1.0, 2.0, (batch, M)), axis=1)
    lam[:, : M // 2] = 1.0 + 1e-10 * rng.uniform(0.0, 1.0, (batch, M // 2))
    Q, _ = np.linalg.qr(rng.standard_normal((batch, M, M)))
    return np.matmul(Q * lam[:, None, :], np.transpose(Q, (0, 2, 1)))


def both_paths(lk, A):
    import torch
    At = torch.from_numpy(np.ascontiguousarray(A)).cuda()
    batch, M, _ = A.shape
    w = torch.full((batch, M), float("nan"), dtype=torch.float64, device="cuda")
    V = torch.full((batch, M, M), float("nan"), dtype=torch.float64, device="cuda")
    info = torch.full((batch,), -1, dtype=torch.int32, device="cuda")
    lk.syev_batched_static(At, w, V, info)
    wr, Vr, ir = lk.syev_batched(At)
    torch.cuda.synchronize()
    return (w.cpu().numpy(), V.cpu().numpy(), info.cpu().numpy()), (wr.cpu().numpy(), Vr.cpu().numpy(), ir.cpu().numpy())


def check(A, got, ref, what):
    w, V, info = got
    wr, Vr, ir = ref
    assert (info == ir).all(), what
    parity.assert_evd(A, w, V, wr, what)                       # residual, orthogonality, eigenvalues vs the existing path
    # same kernels on the same inputs: the eigenvectors agree entry by entry (no sign freedom left)
    assert np.abs(V - Vr).max() <= parity.TOL_ORTH, f"{what}: V {np.abs(V - Vr).max():.3e}"


def test_static_matches_existing_path_on_calls_in_a_row(lk):
    """Calls in a row on the one array, each against letkf_syev_batched: the paper's latency case
    (PAPER.md:323, 256 matrices of M = 64), then a smaller batch of other matrices (stale records of the
    first call behind it), clustered spectra (rotation-log route), another order (another layout of the
    array), an order above the register path, and the first input again."""
    cases = [
        ("config N4", wl.letkf_shaped(256, 64, 98, config_index=3)),
        ("smaller batch", wl.letkf_shaped(100, 64, 98, config_index=7)),
        ("clustered", clustered(64, 64, 5)),
        ("M=33", wl.letkf_shaped(129, 33, 49, config_index=11)),
        ("M=100", wl.letkf_shaped(9, 100, 120, config_index=12)),
        ("config N4 again", wl.letkf_shaped(256, 64, 98, config_index=3)),
    ]
    first = None
    for what, A in cases:
        got, ref = both_paths(lk, A)
        check(A, got, ref, what)
        if what == "config N4":
            first = got
        if what == "config N4 again":                          # and the same bits as the first time
            assert np.array_equal(first[0], got[0]) and np.array_equal(first[1], got[1])


def test_static_takes_no_device_memory(lk):
    import torch
    A = torch.from_numpy(wl.letkf_shaped(200, 48, 49, config_index=5)).cuda()
    w = torch.empty((200, 48), dtype=torch.float64, device="cuda")
    V = torch.empty_like(A)
    lk.syev_batched_static(A, w, V)                            # (first use of these kernels loads them)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        lk.syev_batched_static(A, w, V)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0


def test_static_rejects_what_does_not_fit(lk):
    import torch
    for M in (16, 64, 128):
        nmax = lk.syev_static_max_batch(M)
        assert nmax >= 1
        assert lk.syev_workspace_bytes(M, 1) <= lk.STATIC_WORK_BYTES
        A = torch.zeros((nmax + 1, M, M), dtype=torch.float64, device="cuda")
        w = torch.empty((nmax + 1, M), dtype=torch.float64, device="cuda")
        with pytest.raises(lk.LetkfError, match="static scratch array"):
            lk.syev_batched_static(A, w, A)
    assert lk.syev_static_max_batch(64) >= 256                 # the paper's latency case fits
    assert lk.syev_static_max_batch(0) == 0 and lk.syev_static_max_batch(257) == 0
    # the largest batch that fits runs
    M = 64
    nmax = lk.syev_static_max_batch(M)
    An = wl.letkf_shaped(nmax, M, 98, config_index=9)
    got, ref = both_paths(lk, An)
    check(An, got, ref, "largest batch")

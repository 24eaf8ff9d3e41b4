"""GPU parity: letkf_syev_batched (through the C ABI) against the CPU oracle on the same seeded
inputs.  PAPER.md:142, 183 (EVD by Householder + QL); tolerances of north_star / parity.py."""
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


def run_gpu(lk, A, **kw):
    import torch
    At = torch.from_numpy(np.ascontiguousarray(A)).cuda()
    w, V, info = lk.syev_batched(At, **kw)
    torch.cuda.synchronize()
    return w.cpu().numpy(), V.cpu().numpy(), info.cpu().numpy()


def test_config1_known_spectrum(lk, oracle):
    """BASELINE config 1: M=32, batch=1024, A = Q diag(lam) Q^T; eigenvalues known by construction."""
    A, lam = wl.known_spectrum(batch=1024, M=32)
    w, V, info = run_gpu(lk, A)
    assert (info == 0).all()
    wo, Vo, io, _ = oracle.syev_batched(A)
    assert (io == 0).all()
    parity.assert_evd(A, w, V, wo, "config1 vs oracle")
    scale = lam.max(axis=1)
    assert (np.abs(w - lam).max(axis=1) / scale).max() <= 1e-12      # the construction's own spectrum


@pytest.mark.parametrize("M,p,batch", [(48, 49, 300), (64, 98, 300), (16, 49, 257), (32, 49, 129)])
def test_letkf_shaped_vs_oracle(lk, oracle, M, p, batch):
    """BASELINE configs 2/3/5 (reduced batch): A = ((M-1)/rho) I + Yb^T diag(r) Yb."""
    A = wl.letkf_shaped(batch, M, p, config_index=20 + M)
    w, V, info = run_gpu(lk, A)
    assert (info == 0).all()
    wo, _, _, _ = oracle.syev_batched(A)
    parity.assert_evd(A, w, V, wo, f"M={M} p={p}")


@pytest.mark.parametrize("M", [1, 2, 3, 4, 5, 7, 15, 17, 31, 33, 47, 63, 65, 96, 100, 128])
def test_any_order_vs_oracle(lk, oracle, M):
    batch = 37 if M <= 65 else 9
    rng = np.random.Generator(np.random.Philox(key=77 + M))
    G = rng.standard_normal((batch, M, M))
    A = G + np.transpose(G, (0, 2, 1))
    w, V, info = run_gpu(lk, A)
    assert (info == 0).all()
    wo, _, _, _ = oracle.syev_batched(A)
    parity.assert_evd(A, w, V, wo, f"random symmetric M={M}")


@pytest.mark.parametrize("M", [192, 256])
def test_large_order_vs_oracle(lk, oracle, M):
    A = wl.config5(M, batch=4)
    w, V, info = run_gpu(lk, A)
    assert (info == 0).all()
    wo, _, _, _ = oracle.syev_batched(A)
    parity.assert_evd(A, w, V, wo, f"config5 M={M}")


@pytest.mark.parametrize("p", [0, 3, 48])
def test_paper_shaped_clusters(lk, oracle, p):
    """Dense (l_max=1, V=3 -> p=3) and sparse (p=48) observation
    shapes: an (M-p)-fold eigenvalue cluster at (M-1)/rho and zero Householder columns."""
    M, batch = 64, 64
    A = wl.letkf_shaped(batch, M, p, config_index=600 + p)
    w, V, info = run_gpu(lk, A)
    assert (info == 0).all()
    wo, _, _, _ = oracle.syev_batched(A)
    parity.assert_evd(A, w, V, wo, f"cluster p={p}")
    if p < M - 1:
        assert np.abs(w[:, : M - max(p, 1)] - (M - 1) / wl.RHO).max() <= 1e-12 * np.abs(wo).max()


@pytest.mark.parametrize("M", [8, 64, 100])
def test_toeplitz_closed_form(lk, M):
    """tridiag(1,0,1): lambda_k = 2 cos(k pi/(M+1)) -- closed form, no oracle involved."""
    A = np.stack([wl.toeplitz_tridiagonal(M), wl.toeplitz_tridiagonal(M, a=3.0, b=-0.5)])
    w, V, info = run_gpu(lk, A)
    k = np.arange(1, M + 1)
    exact0 = np.sort(2.0 * np.cos(k * np.pi / (M + 1)))
    exact1 = np.sort(3.0 - 1.0 * np.cos(k * np.pi / (M + 1)))
    assert np.abs(w[0] - exact0).max() <= 1e-12 * 2
    assert np.abs(w[1] - exact1).max() <= 1e-12 * 4
    parity.assert_evd(A, w, V, None, "toeplitz")


def test_degenerate_inputs(lk):
    M = 64
    A = np.zeros((4, M, M))
    A[1] = 3.5 * np.eye(M)                                   # A = cI
    A[2] = np.diag(np.arange(M, 0, -1.0))                    # diagonal, descending
    A[3][0, 0] = 1.0                                         # rank one
    w, V, info = run_gpu(lk, A)
    assert (info == 0).all()
    parity.assert_evd(A, w, V, None, "degenerate")
    assert np.abs(w[0]).max() == 0.0
    assert np.abs(w[1] - 3.5).max() == 0.0
    assert np.abs(w[2] - np.arange(1.0, M + 1)).max() == 0.0


def test_only_lower_triangle_is_read(lk, oracle):
    A = wl.letkf_shaped(40, 64, 98, config_index=31)
    junk = A.copy()
    iu = np.triu_indices(64, 1)
    junk[:, iu[0], iu[1]] = 1e30
    w, V, _ = run_gpu(lk, junk)
    w2, V2, _ = run_gpu(lk, A)
    assert np.array_equal(w, w2) and np.array_equal(V, V2)


def test_in_place_and_user_workspace(lk):
    import torch
    A = wl.letkf_shaped(100, 48, 49, config_index=32)
    At = torch.from_numpy(A).cuda()
    w0, V0, _ = lk.syev_batched(At)
    nbytes = lk.syev_workspace_bytes(48, 100)
    work = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    Ain = At.clone()
    w1, V1, _ = lk.syev_batched(Ain, V=Ain, work=work)
    torch.cuda.synchronize()
    assert V1.data_ptr() == Ain.data_ptr()
    assert torch.equal(w0, w1) and torch.equal(V0, V1)
    small = torch.empty(64, dtype=torch.uint8, device="cuda")
    with pytest.raises(lk.LetkfError):
        lk.syev_batched(At, work=small)


@pytest.mark.parametrize("batch", [1, 31, 33, 1000])
def test_ragged_batches(lk, oracle, batch):
    A = wl.letkf_shaped(batch, 64, 98, config_index=33)
    w, V, info = run_gpu(lk, A)
    assert (info == 0).all()
    sel = np.unique(np.linspace(0, batch - 1, min(batch, 40)).astype(int))
    wo, _, _, _ = oracle.syev_batched(A[sel])
    parity.assert_evd(A[sel], w[sel], V[sel], wo, f"batch={batch}")
    parity.assert_evd(A, w, V, None, f"batch={batch} all")


def test_determinism(lk):
    A = wl.letkf_shaped(200, 64, 98, config_index=34)
    a = run_gpu(lk, A)
    b = run_gpu(lk, A)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_nan_input_terminates(lk):
    A = wl.letkf_shaped(8, 64, 98, config_index=35)
    A[3, 10, 4] = np.nan
    w, V, info = run_gpu(lk, A)
    assert info[3] != 0
    good = [0, 1, 2, 4, 5, 6, 7]
    assert (info[good] == 0).all()
    parity.assert_evd(A[good], w[good], V[good], None, "neighbours of a NaN matrix")


@pytest.mark.parametrize("scale", [1e-138, 1e138])
def test_extreme_scale_takes_the_slow_path(lk, oracle, scale):
    """Matrices scaled so that r2 = f^2 + g^2 of the QL rotation step leaves [1e-280, 1e280]: the
    branch-free fast step only flags them (ql_kernel.cuh) and the slow path, whose step handles the
    rare cases one by one, must redo them -- same tolerances, neighbours untouched.  (Outside the
    documented range 1e-100 < ||A|| < 1e100, but nowhere near under/overflow of the result.)"""
    A = wl.letkf_shaped(96, 64, 98, config_index=39)
    A[1::3] *= scale
    try:
        lk.set_option("bisect", 0)                        # (the QL kernel, as large batches use it)
        w, V, info = run_gpu(lk, A)
    finally:
        lk.set_option("bisect", -1)
    assert ((info & 0xFFFF) == 0).all()
    slow = (info & lk.INFO_SLOWPATH).astype(bool)
    assert slow[1::3].all() and not slow[0::3].any() and not slow[2::3].any()
    wo, _, _, _ = oracle.syev_batched(A)
    parity.assert_evd(A, w, V, wo, f"scale {scale:g}")
    w, V, info = run_gpu(lk, A)                           # small batch: the multisection kernel has no such range
    assert ((info & 0xFFFF) == 0).all()
    parity.assert_evd(A, w, V, wo, f"scale {scale:g}, multisection")


def test_headline_full_size(lk, oracle):
    """BASELINE config 3 at full size (M=64, batch=16384, the launch configuration bench.py times):
    residual/orthogonality/ordering on every matrix, oracle parity on a strided sample."""
    A = wl.config3()
    w, V, info = run_gpu(lk, A)
    assert (info == 0).all()
    for b0 in range(0, A.shape[0], 2048):
        sl = slice(b0, b0 + 2048)
        parity.assert_evd(A[sl], w[sl], V[sl], None, f"config3 [{b0}:]")
    assert np.abs(w[:, 0] - 63 / wl.RHO).max() <= 1e-12 * w.max()   # A 1 = ((M-1)/rho) 1 (rows centred)
    sel = np.arange(0, A.shape[0], 128)
    wo, _, _, _ = oracle.syev_batched(A[sel])
    parity.assert_evd(A[sel], w[sel], V[sel], wo, "config3 sample vs oracle")


def test_config2_full_size(lk, oracle):
    A = wl.config2()
    w, V, info = run_gpu(lk, A)
    assert (info == 0).all()
    for b0 in range(0, A.shape[0], 4096):
        sl = slice(b0, b0 + 4096)
        parity.assert_evd(A[sl], w[sl], V[sl], None, f"config2 [{b0}:]")
    sel = np.arange(0, A.shape[0], 128)
    wo, _, _, _ = oracle.syev_batched(A[sel])
    parity.assert_evd(A[sel], w[sel], V[sel], wo, "config2 sample vs oracle")


@pytest.mark.parametrize("M", [3, 16, 48, 64])
def test_generic_kernels_at_small_order(lk, oracle, M):
    """The any-M kernels (normally M > 64 and the overflow finisher) forced onto small M."""
    A = wl.letkf_shaped(33, M, 49, config_index=70 + M)
    lk.set_option("force_generic", 1)
    try:
        w, V, info = run_gpu(lk, A)
    finally:
        lk.set_option("force_generic", 0)
    assert (info == 0).all()
    wo, _, _, _ = oracle.syev_batched(A)
    parity.assert_evd(A, w, V, wo, f"generic M={M}")


def test_pipelined_equals_single_stream(lk):
    """The sub-chunk pipeline over private streams (Streams) only reorders
    launches: its results are bitwise those of the one-stream, one-chunk run, also in place and
    when the call follows other work on a user stream."""
    import torch
    A = wl.letkf_shaped(4096 + 37, 64, 98, config_index=901)
    At = torch.from_numpy(A).cuda()
    try:
        lk.set_option("pipeline", 0)
        w0, V0, i0 = lk.syev_batched(At)
        torch.cuda.synchronize()
    finally:
        lk.set_option("pipeline", 1)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        B = At.clone()                                   # produced on the user stream just before
        w1, V1, i1 = lk.syev_batched(B, V=B, stream=st)  # in place
        s = V1.sum()                                     # consumed on the user stream just after
    st.synchronize()
    assert torch.equal(w0, w1) and torch.equal(V0, V1) and torch.equal(i0, i1)
    assert torch.isfinite(s)
    assert lk.last_launch_count() >= 4 * 3               # >= 4 sub-chunks x 3 kernels


@pytest.mark.parametrize("pinned", [True, False])
def test_host_entry_point_equals_device_call(lk, pinned):
    """letkf_syev_batched_host (chunked H2D -> kernels -> D2H inside the library) returns bitwise
    what the device call returns, from pinned and from pageable host memory, ragged last chunk."""
    import torch
    A = torch.from_numpy(wl.letkf_shaped(2 * 2048 + 300, 64, 98, config_index=902))
    wd, Vd, idv = lk.syev_batched(A.cuda())
    torch.cuda.synchronize()
    Ah = A.pin_memory() if pinned else A
    w, V, info = lk.syev_batched_host(Ah)
    assert torch.equal(w, wd.cpu()) and torch.equal(V, Vd.cpu()) and torch.equal(info, idv.cpu())
    w2, V2, _ = lk.syev_batched_host(Ah.clone(), V=None)          # second call reuses the streams
    assert torch.equal(V2, V)


@pytest.mark.parametrize("M,batch", [(64, 2100), (48, 300), (100, 12)])
def test_log_overflow_slow_path(lk, oracle, M, batch):
    """With the rotation log shrunk the QL kernel flags matrices whose log would overflow and the
    classic iteration completes them (inside the apply kernel for M <= 64, in the finisher on the
    stored Q above): same tolerances, and info carries LETKF_INFO_SLOWPATH for exactly those
    matrices."""
    A = wl.letkf_shaped(batch, M, 98 if M >= 64 else 49, config_index=930 + M)
    try:
        lk.set_option("log_shrink", 3)
        lk.set_option("evec", 0)                          # (M <= 64: every matrix through the log)
        w, V, info = run_gpu(lk, A)
    finally:
        lk.set_option("log_shrink", 1)
        lk.set_option("evec", 1)
    assert ((info & 0xFFFF) == 0).all()
    assert (info & lk.INFO_SLOWPATH).astype(bool).all(), "every matrix should have taken the slow path"
    wo, _, _, _ = oracle.syev_batched(A[:64])
    parity.assert_evd(A, w, V, None, f"slow path M={M}")
    assert np.abs(w[:64] - wo).max() <= parity.TOL_W * np.abs(wo).max()
    w2, V2, info2 = run_gpu(lk, A)
    assert (info2 == 0).all() and np.abs(w2 - w).max() <= parity.TOL_W * np.abs(w).max()


@pytest.mark.parametrize("M", [9, 16, 21, 48, 64, 100, 160, 200])
def test_hard_spectra(lk, oracle, M):
    """Matrices that stress the tridiagonal eigensolver and the deflation logic: Wilkinson W+ (pairs of
    eigenvalues agreeing to ~1e-14), two of them glued by a tiny coupling, graded matrices over
    many orders of magnitude (up and down), a rank-one update of the identity (an (M-1)-fold
    cluster), a negative-definite matrix, an arrowhead, and entries at both ends of the documented
    range (1e-100 < max|A| < 1e100).  Residual / orthogonality at tolerance, eigenvalues against
    the oracle."""
    rng = np.random.Generator(np.random.Philox(key=4242 + M))
    mats = []
    k = (M - 1) // 2
    Wk = np.diag(np.abs(np.arange(M) - k).astype(float)) + np.diag(np.ones(M - 1), 1) + np.diag(np.ones(M - 1), -1)
    mats.append(Wk)                                                        # Wilkinson W+
    G = Wk.copy(); G[M // 2, M // 2 - 1] = G[M // 2 - 1, M // 2] = 1e-9    # glued halves
    mats.append(G)
    Q, _ = np.linalg.qr(rng.standard_normal((M, M)))
    mats.append(Q @ np.diag(10.0 ** np.linspace(-12, 6, M)) @ Q.T)         # wide spectrum, dense
    s = 10.0 ** np.linspace(0, 8, M)
    B = rng.standard_normal((M, M)); B = B + B.T
    mats.append(B * np.outer(s, s) / s[-1] ** 2)                           # graded downwards
    mats.append((B * np.outer(s, s) / s[-1] ** 2)[::-1, ::-1].copy())      # graded upwards
    u = rng.standard_normal(M)
    mats.append(np.eye(M) + np.outer(u, u))                                # (M-1)-fold cluster at 1
    mats.append(-(B @ B.T) - np.eye(M))                                    # negative definite
    Ar = np.diag(np.arange(1.0, M + 1)); Ar[-1, :-1] = Ar[:-1, -1] = 0.5   # arrowhead
    mats.append(Ar)
    mats.append(B * 1e-99)
    mats.append(B * 1e98)
    A = np.stack([0.5 * (X + X.T) for X in mats])
    w, V, info = run_gpu(lk, A)
    assert (info == 0).all()
    wo, _, io, _ = oracle.syev_batched(A)
    assert (io == 0).all()
    parity.assert_evd(A, w, V, wo, f"hard spectra M={M}")


@pytest.mark.parametrize("mode", [0, 2, 12])
@pytest.mark.parametrize("M", [65, 71, 96, 97, 113, 128, 129, 145, 160])
def test_mid_tridiagonalisation_both_forms(lk, oracle, M, mode):
    """64 < M <= 160 (mid_kernels.cuh): the reduction with the matrix in shared memory
    (mid_reg = 0) and in registers (mid_reg = 2) at every size class (MT = 96 / 128 / 160), ragged
    orders included; the default picks one of the two by size.  Up to M = 128 the register form hands
    its trailing 64 x 64 block to the kernels of the M <= 64 path (mid_split = 1, default; mode 12 here
    is mid_reg = 2 with mid_split = 0: one kernel down to pivot 1).  Low-rank inputs (p = 3 < M - 1)
    exercise the tau = 0 pivots (reading G19) and the eigenvalue cluster."""
    A = np.concatenate([wl.letkf_shaped(9, M, 98, config_index=960 + M),
                        wl.letkf_shaped(4, M, 3, config_index=961 + M)])
    try:
        lk.set_option("mid_reg", mode % 10)
        lk.set_option("mid_split", 0 if mode >= 10 else 1)
        w, V, info = run_gpu(lk, A)
    finally:
        lk.set_option("mid_reg", 1)
        lk.set_option("mid_split", 1)
    assert (info == 0).all()
    wo, _, _, _ = oracle.syev_batched(A)
    parity.assert_evd(A, w, V, wo, f"mid M={M} mid_reg={mode}")


VARIANTS = {"direct": {}, "replay": {"evec": 0}, "qform": {"qform": 1}, "split": {"split": 1}, "pair": {"pair": 1},
            "nopair": {"pair": 0}, "nosplit": {"split": 0}, "nopack": {"pack": 0}, "nopack_replay": {"pack": 0, "evec": 0},
            "pack_tridiag": {"pack": 2}, "pack_apply": {"pack": 3}}


@pytest.mark.parametrize("variant", sorted(VARIANTS))
@pytest.mark.parametrize("M,p", [(64, 98), (57, 98), (48, 49), (33, 49), (16, 49), (5, 49), (64, 3), (64, 48), (64, 0)])
def test_register_path_variants(lk, oracle, M, p, variant):
    """The three forms of the M <= 64 path.  "direct" (default): the reduction
    kernel keeps the reflectors, the QL kernel finds the eigenvalues and classifies the matrix, the
    apply kernel forms the eigenvectors of T by twisted factorisations where the spectrum allows
    (else it replays the logged rotations on the identity) and does the back-transform
    V = H_{M-1} ... H_1 Z.  "replay" (evec = 0): always the logged rotations.  "qform" (qform = 1):
    the explicit Q is formed by the reduction kernel and the rotations are replayed on its rows.
    "split" (split = 1, acts for 48 < M <= 64): the reduction as two kernels.  "pair" / "nopair"
    (32 < M <= 64): two matrices per CTA of the reduction kernel, or one (odd batch: a CTA with one).
    Each also with the rotation log shrunk, which sends the replaying matrices to the classic
    iteration inside the apply kernel."""
    A = wl.letkf_shaped(151, M, p, config_index=990 + M + p)       # (odd: the paired kernel ends on a CTA with one matrix)
    try:
        for k, v in VARIANTS[variant].items():
            lk.set_option(k, v)
        w, V, info = run_gpu(lk, A)
        lk.set_option("log_shrink", 4)
        w2, V2, info2 = run_gpu(lk, A)
    finally:
        for k, v in (("qform", 0), ("evec", 1), ("log_shrink", 1), ("split", 1), ("pair", -1), ("pack", 1)):
            lk.set_option(k, v)
    assert (info == 0).all()
    wo, _, _, _ = oracle.syev_batched(A)
    parity.assert_evd(A, w, V, wo, f"{variant} M={M}")
    parity.assert_evd(A, w2, V2, wo, f"{variant}, log shrunk, M={M}")
    assert ((info2 & 0xFFFF) == 0).all()
    if p >= M - 1 and M >= 16 and variant in ("replay", "qform", "nopack_replay"):
        assert (info2 & lk.INFO_SLOWPATH).astype(bool).all()


@pytest.mark.parametrize("mode", ["direct", "replay", "slow"])
@pytest.mark.parametrize("M", [2, 3, 7, 8, 9, 10, 13, 15, 16])
def test_two_matrices_per_warp(lk, oracle, M, mode):
    """M <= 16 (pack_kernels.cuh): two matrices share a warp in the reduction and in the
    apply kernel.  A batch that mixes, matrix by matrix, LETKF-shaped inputs, low-rank ones (repeated
    eigenvalue, tau = 0 pivots), a diagonal matrix, the Wilkinson matrix and a glued pair of them, a
    graded matrix and an (M-1)-fold cluster -- so the two halves of a warp take different routes
    through the apply kernel -- at batch sizes that leave the last half warp, warp and CTA ragged;
    with the eigenvector route (default), every matrix through the rotation log (evec = 0), and the
    log shrunk (classic iteration inside the apply kernel).  Same tolerances as everywhere."""
    rng = np.random.Generator(np.random.Philox(key=5150 + M))
    k = (M - 1) // 2
    Wk = np.diag(np.abs(np.arange(M) - k).astype(float)) + np.diag(np.ones(M - 1), 1) + np.diag(np.ones(M - 1), -1)
    G = Wk.copy()
    if M >= 4:
        G[M // 2, M // 2 - 1] = G[M // 2 - 1, M // 2] = 1e-9
    B = rng.standard_normal((M, M)); B = B + B.T
    s = 10.0 ** np.linspace(0, 8, M)
    u = rng.standard_normal(M)
    special = [Wk, G, np.diag(np.arange(1.0, M + 1)), B * np.outer(s, s) / s[-1] ** 2, np.eye(M) + np.outer(u, u),
               -(B @ B.T) - np.eye(M), 3.0 * np.eye(M)]
    for batch in (1, 2, 7, 8, 9, 203):
        A = wl.letkf_shaped(batch, M, 49, config_index=1200 + M + batch)
        A[1::5] = wl.letkf_shaped(len(A[1::5]), M, 3, config_index=1300 + M)      # low rank: an (M-3)-fold eigenvalue
        for i in range(2, batch, 3):
            A[i] = special[(i // 3) % len(special)]
        try:
            if mode != "direct":
                lk.set_option("evec", 0)
            if mode == "slow":
                lk.set_option("log_shrink", 4)
            w, V, info = run_gpu(lk, A)
        finally:
            lk.set_option("evec", 1)
            lk.set_option("log_shrink", 1)
        assert ((info & 0xFFFF) == 0).all()
        wo, _, io, _ = oracle.syev_batched(A)
        assert (io == 0).all()
        parity.assert_evd(A, w, V, wo, f"packed M={M} batch={batch} {mode}")


@pytest.mark.parametrize("force", [0, 1])
@pytest.mark.parametrize("M,p", [(64, 98), (57, 98), (48, 49), (33, 49), (16, 49), (5, 49), (2, 7), (64, 3), (64, 48), (64, 0)])
def test_eigenvalues_by_multisection(lk, oracle, M, p, force):
    """The latency-regime eigenvalue kernel (bisect_kernel.cuh: M threads per matrix,
    multisection on the Sturm count) against the QL kernel's one thread per matrix: small batches take
    it by default, letkf_set_option("bisect", 0 / 1) forces either.  Both feed the same classifier
    and the same apply kernel; clustered spectra (p = 3, 48) go on to the logging QL pass, shifted by
    the eigenvalues found here."""
    A = wl.letkf_shaped(130, M, p, config_index=1100 + M + p)
    try:
        lk.set_option("bisect", force)
        w, V, info = run_gpu(lk, A)
    finally:
        lk.set_option("bisect", -1)
    assert (info == 0).all()
    wo, _, _, _ = oracle.syev_batched(A)
    parity.assert_evd(A, w, V, wo, f"bisect={force} M={M} p={p}")


def test_direct_eigenvectors_are_used_and_fall_back(lk, oracle):
    """Which matrices take which route: well separated spectra (config 3) need no rotation at all
    (the profile counts none); a spectrum with eigenvalues closer than 1e-8 ||T|| inside one
    unreduced block (Wilkinson's W21+, pairs agreeing to 1e-14) has its rotations logged and
    replayed; both meet the tolerances."""
    import torch
    A = wl.letkf_shaped(256, 64, 98, config_index=3)
    k = 10
    Wk = np.diag(np.abs(np.arange(21) - k).astype(float)) + np.diag(np.ones(20), 1) + np.diag(np.ones(20), -1)
    B = np.stack([Wk] * 40)
    for X, expect_rot in ((A, False), (B, True)):
        Xt = torch.from_numpy(X).cuda()
        lk.profile_enable(1)
        try:
            w, V, info = lk.syev_batched(Xt)
            torch.cuda.synchronize()
            nrot = lk.profile_rotations()
        finally:
            lk.profile_enable(0)
        assert int(info.abs().max()) == 0
        assert (nrot > 0) == expect_rot
        wo, _, _, _ = oracle.syev_batched(X)
        parity.assert_evd(X, w.cpu().numpy(), V.cpu().numpy(), wo, "direct / replay routes")


@pytest.mark.parametrize("bigvec", [1, 0])
@pytest.mark.parametrize("M,p", [(65, 98), (80, 49), (96, 98), (97, 200), (128, 98), (128, 3), (130, 300), (160, 98), (161, 98),
                                 (192, 98), (200, 400), (255, 98), (256, 98), (256, 512)])
def test_eigenvector_route_above_64(lk, oracle, M, p, bigvec):
    """M > 64 (big_kernels.cuh): where the classifier allows, the eigenvectors of T by twisted
    factorisations (one thread per eigenvector, the vector in the matrix's record of the rotation
    log) and V = Q Z as one product on the FP64 tensor cores; letkf_set_option("bigvec", 0) sends
    every matrix through the rotation log as before.  Shapes: full rank (p >= M - 1: every
    eigenvalue simple), the sweep's p = 98 < M - 1 (an (M - 98)-fold eigenvalue: T falls apart into
    1 x 1 blocks there -- reading G24), p = 3, ragged orders at every tile shape of the product;
    the LETKF-shaped workloads must take the new route (no rotation logged) and the hard spectra of
    test_hard_spectra (which run with the default) must not."""
    import torch
    batch = 21 if M <= 160 else 9
    A = wl.letkf_shaped(batch, M, p, config_index=1400 + M + p)
    lk.profile_enable(1)
    try:
        lk.set_option("bigvec", bigvec)
        w, V, info = lk.syev_batched(torch.from_numpy(A).cuda())
        torch.cuda.synchronize()
        nrot, ndirect = lk.profile_rotations(), lk.profile_direct()
    finally:
        lk.set_option("bigvec", 1)
        lk.profile_enable(0)
    w, V, info = w.cpu().numpy(), V.cpu().numpy(), info.cpu().numpy()
    assert (info == 0).all()
    if bigvec and p >= M - 1:
        assert ndirect == batch and nrot == 0, f"{ndirect} of {batch} matrices on the eigenvector route, {nrot} rotations"
    if not bigvec:
        assert nrot > 0
    wo, _, _, _ = oracle.syev_batched(A)
    parity.assert_evd(A, w, V, wo, f"M={M} p={p} bigvec={bigvec}")


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("M,p", [(64, 98), (57, 98), (33, 49), (16, 49), (64, 3), (96, 98), (200, 98)])
def test_ql_one_and_two_pass(lk, oracle, M, p, mode):
    """letkf_set_option("two_pass", 0 / 1): the QL iteration logged in one pass (Wilkinson shifts) or
    with a second pass shifted by the eigenvalues of the first: both are
    orthogonal similarities of the same tridiagonal matrix -- same tolerances.  By default the
    batch size picks one (large batches: two passes)."""
    A = wl.letkf_shaped(150 if M <= 64 else 7, M, p, config_index=940 + M + p)
    try:
        lk.set_option("two_pass", mode)
        lk.set_option("bigvec", 0)                        # (M > 64: every matrix through the log)
        w, V, info = run_gpu(lk, A)
    finally:
        lk.set_option("two_pass", -1)
        lk.set_option("bigvec", 1)
    assert (info == 0).all()
    wo, _, _, _ = oracle.syev_batched(A)
    parity.assert_evd(A, w, V, wo, f"two_pass={mode} M={M}")


@pytest.mark.parametrize("M,batch,sub,slots", [(64, 1000, 64, 2), (32, 777, 128, 3), (100, 150, 32, 2), (64, 4133, 0, 0)])
def test_workspace_ring(lk, oracle, M, batch, sub, slots):
    """The sub-chunk pipeline keeps `slots` sub-chunks in flight, each in a slot of the workspace that
    the next tenant takes over when its last kernel is done (Streams).  With a
    small sub-chunk and few slots every slot is reused many times: results must equal the
    one-stream run bitwise (ragged last sub-chunk included)."""
    import torch
    A = wl.letkf_shaped(batch, M, 98 if M >= 64 else 49, config_index=970 + M)
    At = torch.from_numpy(A).cuda()
    try:
        lk.set_option("two_pass", 1)
        lk.set_option("pipeline", 0)
        w0, V0, i0 = lk.syev_batched(At)
        torch.cuda.synchronize()
        lk.set_option("pipeline", 1)
        lk.set_option("sub_chunk", sub)
        lk.set_option("slots", slots)
        work = torch.empty(lk.syev_workspace_bytes(M, batch), dtype=torch.uint8, device="cuda")
        w1, V1, i1 = lk.syev_batched(At, work=work)
        w2, V2, i2 = lk.syev_batched(At, work=work)      # back to back on the same workspace
        torch.cuda.synchronize()
    finally:
        for k, v in (("pipeline", 1), ("sub_chunk", 0), ("slots", 0), ("two_pass", -1)):
            lk.set_option(k, v)
    assert int(i1.abs().max()) == 0
    assert torch.equal(w0, w1) and torch.equal(V0, V1) and torch.equal(w0, w2) and torch.equal(V0, V2)
    sel = slice(0, 48)
    wo, _, _, _ = oracle.syev_batched(A[sel])
    parity.assert_evd(A[sel], w1[sel].cpu().numpy(), V1[sel].cpu().numpy(), wo, f"ring M={M}")


def test_workspace_smaller_than_recommended(lk):
    """Any workspace that holds at least one matrix is accepted: the call then keeps fewer
    sub-chunks in flight, or runs chunk after chunk on the caller's stream; one that holds none is
    refused (argument 7)."""
    import torch
    A = torch.from_numpy(wl.letkf_shaped(3000, 64, 98, config_index=975)).cuda()
    w0, V0, _ = lk.syev_batched(A)
    full = lk.syev_workspace_bytes(64, 3000)
    for frac in (0.5, 0.1):
        work = torch.empty(int(full * frac), dtype=torch.uint8, device="cuda")
        lib = lk.load()
        import ctypes
        w = torch.empty_like(w0); V = torch.empty_like(V0); info = torch.zeros(3000, dtype=torch.int32, device="cuda")
        st = lib.letkf_syev_batched(ctypes.c_void_p(A.data_ptr()), 64, 3000, ctypes.c_void_p(w.data_ptr()),
                                    ctypes.c_void_p(V.data_ptr()), ctypes.c_void_p(info.data_ptr()),
                                    ctypes.c_void_p(work.data_ptr()), work.numel(),
                                    ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))
        assert st == 0
        torch.cuda.synchronize()
        assert torch.equal(w, w0) and torch.equal(V, V0)
    tiny = torch.empty(1024, dtype=torch.uint8, device="cuda")
    st = lib.letkf_syev_batched(ctypes.c_void_p(A.data_ptr()), 64, 3000, ctypes.c_void_p(w.data_ptr()),
                                ctypes.c_void_p(V.data_ptr()), ctypes.c_void_p(info.data_ptr()),
                                ctypes.c_void_p(tiny.data_ptr()), 1024,
                                ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert st == -7


def test_host_entry_point_in_passes(lk, oracle):
    """The host entry points process a batch that exceeds the staging arena in passes
    (letkf_set_option("host_pass", n) forces small ones): three passes with a ragged last one, arena
    and workspace reused pass after pass."""
    import torch
    A = torch.from_numpy(wl.letkf_shaped(2 * 1100 + 311, 64, 98, config_index=976))
    try:
        lk.set_option("host_pass", 1100)
        lk.set_option("two_pass", 1)
        lk.set_option("bisect", 0)                        # (the ragged last pass is small: same kernels as the device call)
        w, V, info = lk.syev_batched_host(A.pin_memory())
        wd, Vd, _ = lk.syev_batched(A.cuda())
        torch.cuda.synchronize()
    finally:
        lk.set_option("host_pass", 0)
        lk.set_option("two_pass", -1)
        lk.set_option("bisect", -1)
    assert int(info.abs().max()) == 0
    assert torch.equal(w, wd.cpu()) and torch.equal(V, Vd.cpu())


def test_two_host_threads(lk, oracle):
    """The library keeps its streams, events and staging arena per host thread and snapshots the
    options once per call: two threads drive it at the same time on streams of their own (one the
    EVD, one the fused analysis) while the main thread flips an option the calls must not see
    half-way (a call that changed path between its stages would return garbage)."""
    import threading
    import torch
    A = torch.from_numpy(wl.letkf_shaped(3000, 64, 98, config_index=977)).cuda()
    inp = wl.analysis_inputs(batch=2500, M=64, p=98, nstate=9, config_index=978)
    t = {k: torch.from_numpy(inp[k]).cuda() for k in ("Yb", "d", "rinv_loc", "Xb")}
    w0, V0, _ = lk.syev_batched(A)
    Xa0 = lk.analysis_batched(t["Yb"], t["d"], t["rinv_loc"], t["Xb"], inp["rho"])["Xa"]
    torch.cuda.synchronize()
    out, err = {}, []

    def evd():
        try:
            st = torch.cuda.Stream()
            for _ in range(6):
                out["evd"] = lk.syev_batched(A, stream=st)
            st.synchronize()
        except Exception as ex:      # pragma: no cover
            err.append(ex)

    def ana():
        try:
            st = torch.cuda.Stream()
            for _ in range(6):
                out["ana"] = lk.analysis_batched(t["Yb"], t["d"], t["rinv_loc"], t["Xb"], inp["rho"], stream=st)
            st.synchronize()
        except Exception as ex:      # pragma: no cover
            err.append(ex)

    th = [threading.Thread(target=evd), threading.Thread(target=ana)]
    for x in th:
        x.start()
    for k in range(400):                                  # an option that switches the kernel family and the
        lk.set_option("force_generic", k & 1)             # meaning of the V buffer between the stages
    for x in th:
        x.join()
    lk.set_option("force_generic", 0)
    assert not err, err
    # each call ran entirely on one path or the other: valid to tolerance either way
    w1, V1, i1 = out["evd"]
    assert int(i1.abs().max()) == 0
    Af = torch.tril(A) + torch.tril(A, -1).transpose(1, 2)
    R = torch.matmul(Af, V1) - V1 * w1.unsqueeze(1)
    assert float((R.flatten(1).norm(dim=1) / Af.flatten(1).norm(dim=1)).max()) <= parity.TOL_RES
    G = torch.matmul(V1.transpose(1, 2), V1) - torch.eye(64, dtype=torch.float64, device="cuda")
    assert float(G.abs().max()) <= parity.TOL_ORTH
    assert float((w1 - w0).abs().max() / w0.abs().max()) <= parity.TOL_W
    Xa1 = out["ana"]["Xa"]
    xbar = t["Xb"].mean(dim=2, keepdim=True)
    num = (Xa1 - Xa0).flatten(1).norm(dim=1)
    den = (Xa0 - xbar).flatten(1).norm(dim=1)
    assert float((num / den).max()) <= parity.TOL_ANALYSIS


@pytest.mark.parametrize("M", [16, 32, 96, 128, 192, 256])
def test_config5_full_sizes(lk, oracle, M):
    """BASELINE config 5 at the sizes bench.py's sweep times (batch = floor(2^26 / M^2)): residual,
    orthogonality and ordering on EVERY matrix (evaluated on the GPU with torch fp64 batched
    matmuls: properties that hold at any size), eigenvalues against the oracle on a strided sample.
    M = 48 and 64 have their own full-size tests (configs 2 and 3)."""
    import torch
    B = (1 << 26) // (M * M)
    A = wl.config5(M, batch=B)
    At = torch.from_numpy(A).cuda()
    w, V, info = lk.syev_batched(At)
    torch.cuda.synchronize()
    assert int(info.abs().max()) == 0
    assert bool((w[:, 1:] >= w[:, :-1]).all())
    L = torch.tril(At)
    Af = L + torch.tril(At, -1).transpose(1, 2)
    step = max(1, B // 16)
    worst_res = worst_orth = 0.0
    for b0 in range(0, B, step):
        sl = slice(b0, min(B, b0 + step))
        R = torch.matmul(Af[sl], V[sl]) - V[sl] * w[sl].unsqueeze(1)
        worst_res = max(worst_res, float((R.flatten(1).norm(dim=1) / Af[sl].flatten(1).norm(dim=1)).max()))
        G = torch.matmul(V[sl].transpose(1, 2), V[sl]) - torch.eye(M, dtype=torch.float64, device="cuda")
        worst_orth = max(worst_orth, float(G.abs().max()))
    assert worst_res <= parity.TOL_RES, f"residual {worst_res:.3e}"
    assert worst_orth <= parity.TOL_ORTH, f"orthogonality {worst_orth:.3e}"
    sel = np.unique(np.linspace(0, B - 1, 12 if M <= 128 else 4).astype(int))
    wo, _, _, _ = oracle.syev_batched(A[sel])
    wg = w[torch.from_numpy(sel).cuda()].cpu().numpy()
    assert (np.abs(wg - wo).max(axis=1) / np.abs(wo).max(axis=1)).max() <= parity.TOL_W


@pytest.mark.parametrize("M,B,p", [(177, 650, 98), (255, 600, 300), (161, 700, 40)])
def test_any_m_path_pipelined_odd_orders(lk, oracle, M, B, p):
    """The any-M kernels (M > 160) in the pipelined regime with odd orders and a ragged last sub-chunk
    (sub-chunks of 296 matrices): the symmetric-half reduction with its full diagonal blocks, the grouped
    Q formation and the prefetching replay see rows and columns that are no multiple of 8 or 32; p above
    M - 1 (no repeated eigenvalue), at the sweep's 98 and well below it (most of T falls apart).  Residual,
    orthogonality and ordering on every matrix, eigenvalues against the oracle on a sample."""
    import torch
    A = wl.letkf_shaped(B, M, p, 700 + M)
    At = torch.from_numpy(A).cuda()
    w, V, info = lk.syev_batched(At)
    torch.cuda.synchronize()
    assert int(info.abs().max()) == 0
    assert bool((w[:, 1:] >= w[:, :-1]).all())
    Af = torch.tril(At) + torch.tril(At, -1).transpose(1, 2)
    R = torch.matmul(Af, V) - V * w.unsqueeze(1)
    res = float((R.flatten(1).norm(dim=1) / Af.flatten(1).norm(dim=1)).max())
    G = torch.matmul(V.transpose(1, 2), V) - torch.eye(M, dtype=torch.float64, device="cuda")
    assert res <= parity.TOL_RES, f"residual {res:.3e}"
    assert float(G.abs().max()) <= parity.TOL_ORTH, f"orthogonality {float(G.abs().max()):.3e}"
    sel = np.array([0, 295, 296, B - 1])
    wo, _, _, _ = oracle.syev_batched(A[sel])
    wg = w[torch.from_numpy(sel).cuda()].cpu().numpy()
    assert (np.abs(wg - wo).max(axis=1) / np.abs(wo).max(axis=1)).max() <= parity.TOL_W

"""Thin Python binding of libletkf (include/letkf.h): argument marshalling only.

Every step of the hot path runs inside the CUDA library; torch is used for device memory and
streams.  There is no CPU fallback: if libletkf.so is missing or no CUDA device is present the
calls raise.  Names and argument order follow the C ABI one to one.
"""
import ctypes
import os

# The sub-chunk pipeline of a call forks onto up to 22 private streams (2 tridiag, 4 apply, 16 QL);
# with the default of 8 hardware work queues, streams that share a queue serialise.  Only effective
# if set before the CUDA context is created, and never overrides the caller's own setting.
os.environ.setdefault("CUDA_DEVICE_MAX_CONNECTIONS", "32")

import torch  # noqa: E402

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libletkf.so")
MAX_M = 256
INFO_SLOWPATH = 0x40000000
INFO_NS_NOCONV = 0x20000000
STATIC_WORK_BYTES = 32 << 20
ERR_STATIC_CAPACITY = -100

EXPORTS = (
    "letkf_syev_batched", "letkf_syev_workspace_bytes",
    "letkf_syev_batched_static", "letkf_syev_static_max_batch",
    "letkf_syev_batched_f32", "letkf_syev_f32_workspace_bytes",
    "letkf_analysis_batched", "letkf_analysis_workspace_bytes", "letkf_analysis_batched_evdfree",
    "letkf_syev_batched_host", "letkf_analysis_batched_host", "letkf_host_release",
    "letkf_analysis_grid", "letkf_analysis_grid_workspace_bytes", "letkf_analysis_grid_host",
    "letkf_probe_dfma", "letkf_last_launch_count",
    "letkf_profile_enable", "letkf_profile_count", "letkf_profile_record", "letkf_profile_record_start", "letkf_profile_rotations", "letkf_profile_direct",
    "letkf_set_option", "letkf_status_string", "letkf_version",
)

_lib = None


class LetkfError(RuntimeError):
    pass


def load():
    """dlopen libletkf.so and declare the prototypes.  Raises if the library is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise LetkfError(
            f"{LIB_PATH} not found: build it with `python -m paper_2308_03310_b200.build` "
            "(or __graft_entry__.build()). There is no CPU fallback.")
    lib = ctypes.CDLL(LIB_PATH)
    vp, ci, cd, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    lib.letkf_syev_batched.argtypes = [vp, ci, ci, vp, vp, vp, vp, sz, vp]
    lib.letkf_syev_batched.restype = ci
    lib.letkf_syev_workspace_bytes.argtypes = [ci, ci]
    lib.letkf_syev_workspace_bytes.restype = sz
    lib.letkf_syev_batched_static.argtypes = [vp, ci, ci, vp, vp, vp, vp]
    lib.letkf_syev_batched_static.restype = ci
    lib.letkf_syev_static_max_batch.argtypes = [ci]
    lib.letkf_syev_static_max_batch.restype = ci
    lib.letkf_syev_batched_f32.argtypes = [vp, ci, ci, vp, vp, vp, vp, sz, vp]
    lib.letkf_syev_batched_f32.restype = ci
    lib.letkf_syev_f32_workspace_bytes.argtypes = [ci, ci]
    lib.letkf_syev_f32_workspace_bytes.restype = sz
    lib.letkf_analysis_batched.argtypes = [vp, vp, vp, vp, ci, ci, ci, ci, cd,
                                           vp, vp, vp, vp, vp, sz, vp]
    lib.letkf_analysis_batched.restype = ci
    lib.letkf_analysis_batched_evdfree.argtypes = [vp, vp, vp, vp, ci, ci, ci, ci, cd, vp, vp, vp, vp, vp]
    lib.letkf_analysis_batched_evdfree.restype = ci
    lib.letkf_analysis_workspace_bytes.argtypes = [ci, ci, ci, ci]
    lib.letkf_analysis_workspace_bytes.restype = sz
    lib.letkf_syev_batched_host.argtypes = [vp, ci, ci, vp, vp, vp]
    lib.letkf_syev_batched_host.restype = ci
    lib.letkf_analysis_batched_host.argtypes = [vp, vp, vp, vp, ci, ci, ci, ci, cd, vp, vp, vp, vp]
    lib.letkf_analysis_batched_host.restype = ci
    lib.letkf_analysis_grid.argtypes = [vp, vp, vp, vp, ci, ci, ci, ci, ci, ci, ci, cd, cd, cd, vp, vp, vp, vp, sz, vp]
    lib.letkf_analysis_grid.restype = ci
    lib.letkf_analysis_grid_workspace_bytes.argtypes = [ci, ci, ci, ci, ci, ci]
    lib.letkf_analysis_grid_workspace_bytes.restype = sz
    lib.letkf_analysis_grid_host.argtypes = [vp, vp, vp, vp, ci, ci, ci, ci, ci, ci, ci, cd, cd, cd, vp, vp, vp]
    lib.letkf_analysis_grid_host.restype = ci
    lib.letkf_host_release.argtypes = []
    lib.letkf_host_release.restype = None
    lib.letkf_probe_dfma.argtypes = [vp, ci, ci, ci, ctypes.POINTER(ctypes.c_ulonglong), vp]
    lib.letkf_probe_dfma.restype = ci
    lib.letkf_last_launch_count.argtypes = []
    lib.letkf_last_launch_count.restype = ci
    lib.letkf_profile_enable.argtypes = [ci]
    lib.letkf_profile_enable.restype = ci
    lib.letkf_profile_count.argtypes = []
    lib.letkf_profile_count.restype = ci
    lib.letkf_profile_record.argtypes = [ci, ctypes.POINTER(ctypes.c_char_p), ctypes.POINTER(ctypes.c_float)]
    lib.letkf_profile_record.restype = ci
    lib.letkf_profile_record_start.argtypes = [ci, ctypes.POINTER(ctypes.c_float)]
    lib.letkf_profile_record_start.restype = ci
    lib.letkf_profile_rotations.argtypes = []
    lib.letkf_profile_rotations.restype = ctypes.c_longlong
    lib.letkf_profile_direct.argtypes = []
    lib.letkf_profile_direct.restype = ctypes.c_longlong
    lib.letkf_set_option.argtypes = [ctypes.c_char_p, ci]
    lib.letkf_set_option.restype = ci
    lib.letkf_status_string.argtypes = [ci]
    lib.letkf_status_string.restype = ctypes.c_char_p
    lib.letkf_version.argtypes = []
    lib.letkf_version.restype = ci
    _lib = lib
    return lib


def _check(status, what):
    if status != 0:
        msg = load().letkf_status_string(status).decode()
        raise LetkfError(f"{what} failed with status {status}: {msg}")


def _ptr(t):
    return ctypes.c_void_p(t.data_ptr()) if t is not None else ctypes.c_void_p(0)


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def _dev_f64(t, name):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64
            and t.is_contiguous()):
        raise LetkfError(f"{name} must be a contiguous float64 CUDA tensor")
    return t


def _out(t, name, shape, dev, dtype=torch.float64):
    """A caller-supplied output: right device, dtype, exact shape, contiguous."""
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.device == dev and t.dtype == dtype
            and t.is_contiguous() and tuple(t.shape) == tuple(shape)):
        raise LetkfError(f"{name} must be a contiguous {dtype} CUDA tensor of shape {tuple(shape)} on {dev}")
    return t


def _work(work, dev, need):
    if work is None:
        return 0
    if not (isinstance(work, torch.Tensor) and work.is_cuda and work.device == dev and work.is_contiguous()):
        raise LetkfError(f"work must be a contiguous CUDA tensor on {dev}")
    return work.numel() * work.element_size()      # (the library checks the size: smaller ones are legal)


def version():
    return load().letkf_version()


def last_launch_count():
    return load().letkf_last_launch_count()


def syev_workspace_bytes(M, batch):
    return load().letkf_syev_workspace_bytes(M, batch)


def analysis_workspace_bytes(M, p, nstate, batch):
    return load().letkf_analysis_workspace_bytes(M, p, nstate, batch)


def syev_batched(A, w=None, V=None, info=None, work=None, stream=None):
    """letkf_syev_batched: A[batch][M][M] (lower triangle read) -> (w, V, info).

    ``V`` may be ``A`` itself (in place).  Outputs are allocated when not given.  The call is
    stream-ordered and does not synchronise.
    """
    lib = load()
    _dev_f64(A, "A")
    batch, M, M2 = A.shape
    if M != M2:
        raise LetkfError("A must be [batch][M][M]")
    if w is None:
        w = torch.empty((batch, M), dtype=torch.float64, device=A.device)
    if V is None:
        V = torch.empty_like(A)
    if info is None:
        info = torch.zeros((batch,), dtype=torch.int32, device=A.device)
    _out(w, "w", (batch, M), A.device)
    _out(V, "V", (batch, M, M), A.device)
    _out(info, "info", (batch,), A.device, torch.int32)
    wb = _work(work, A.device, lib.letkf_syev_workspace_bytes(M, batch) if batch else 0)
    with torch.cuda.device(A.device):
        st = lib.letkf_syev_batched(_ptr(A), M, batch, _ptr(w), _ptr(V), _ptr(info),
                                    _ptr(work), wb, _stream(stream))
    _check(st, "letkf_syev_batched")
    return w, V, info


def syev_static_max_batch(M):
    return load().letkf_syev_static_max_batch(M)


def syev_batched_static(A, w, V, info=None, stream=None):
    """letkf_syev_batched_static: the EVD with the kernels' scratch memory in the library's static
    device array -- no allocation on the way, so the outputs ``w`` and ``V`` (``V`` may be ``A``) are
    the caller's, ``info`` too where wanted.  batch <= syev_static_max_batch(M), else LetkfError
    (status ERR_STATIC_CAPACITY).  Calls of one device share the array: keep them on one stream."""
    lib = load()
    _dev_f64(A, "A")
    batch, M, M2 = A.shape
    if M != M2:
        raise LetkfError("A must be [batch][M][M]")
    _out(w, "w", (batch, M), A.device)
    _out(V, "V", (batch, M, M), A.device)
    if info is not None:
        _out(info, "info", (batch,), A.device, torch.int32)
    with torch.cuda.device(A.device):
        st = lib.letkf_syev_batched_static(_ptr(A), M, batch, _ptr(w), _ptr(V), _ptr(info), _stream(stream))
    _check(st, "letkf_syev_batched_static")
    return w, V, info


def syev_f32_workspace_bytes(M, batch):
    return load().letkf_syev_f32_workspace_bytes(M, batch)


def syev_batched_f32(A, w=None, V=None, info=None, work=None, stream=None):
    """letkf_syev_batched_f32: the EVD in the paper's precision, A[batch][M][M] float32, M <= 64
    -> (w, V, info) with w, V float32.  ``V`` may be ``A`` itself."""
    lib = load()
    if not (isinstance(A, torch.Tensor) and A.is_cuda and A.dtype == torch.float32 and A.is_contiguous()):
        raise LetkfError("A must be a contiguous float32 CUDA tensor")
    batch, M, M2 = A.shape
    if M != M2:
        raise LetkfError("A must be [batch][M][M]")
    if w is None:
        w = torch.empty((batch, M), dtype=torch.float32, device=A.device)
    if V is None:
        V = torch.empty_like(A)
    if info is None:
        info = torch.zeros((batch,), dtype=torch.int32, device=A.device)
    _out(w, "w", (batch, M), A.device, torch.float32)
    _out(V, "V", (batch, M, M), A.device, torch.float32)
    _out(info, "info", (batch,), A.device, torch.int32)
    wb = _work(work, A.device, 0)
    with torch.cuda.device(A.device):
        st = lib.letkf_syev_batched_f32(_ptr(A), M, batch, _ptr(w), _ptr(V), _ptr(info), _ptr(work), wb, _stream(stream))
    _check(st, "letkf_syev_batched_f32")
    return w, V, info


def analysis_batched(Yb, d, rinv_loc, Xb, rho, Xa=None, want_W=False, want_wbar=False,
                     W=None, wbar=None, info=None, work=None, stream=None):
    """letkf_analysis_batched: Yb[batch][p][M], d[batch][p], rinv_loc[batch][p],
    Xb[batch][nstate][M] -> dict(Xa, W, wbar, info).  ``Xa`` may be ``Xb`` (in place)."""
    lib = load()
    _dev_f64(Yb, "Yb")
    _dev_f64(d, "d")
    _dev_f64(rinv_loc, "rinv_loc")
    _dev_f64(Xb, "Xb")
    batch, p, M = Yb.shape
    nstate = Xb.shape[1]
    if d.shape != (batch, p) or rinv_loc.shape != (batch, p) or Xb.shape != (batch, nstate, M):
        raise LetkfError("inconsistent shapes")
    dev = Xb.device
    if Xa is None:
        Xa = torch.empty_like(Xb)
    if W is None and want_W:
        W = torch.empty((batch, M, M), dtype=torch.float64, device=dev)
    if wbar is None and want_wbar:
        wbar = torch.empty((batch, M), dtype=torch.float64, device=dev)
    if info is None:
        info = torch.zeros((batch,), dtype=torch.int32, device=dev)
    _out(Xa, "Xa", (batch, nstate, M), dev)
    if W is not None:
        _out(W, "W", (batch, M, M), dev)
    if wbar is not None:
        _out(wbar, "wbar", (batch, M), dev)
    _out(info, "info", (batch,), dev, torch.int32)
    wb = _work(work, dev, lib.letkf_analysis_workspace_bytes(M, p, nstate, batch) if batch else 0)
    with torch.cuda.device(dev):
        st = lib.letkf_analysis_batched(_ptr(Yb), _ptr(d), _ptr(rinv_loc), _ptr(Xb),
                                        M, p, nstate, batch, float(rho),
                                        _ptr(Xa), _ptr(W), _ptr(wbar), _ptr(info),
                                        _ptr(work), wb, _stream(stream))
    _check(st, "letkf_analysis_batched")
    return dict(Xa=Xa, W=W, wbar=wbar, info=info)


def analysis_batched_evdfree(Yb, d, rinv_loc, Xb, rho, Xa=None, want_W=False, want_wbar=False, info=None, stream=None):
    """letkf_analysis_batched_evdfree: the analysis by a coupled Newton-Schulz iteration on the FP64
    tensor cores instead of an EVD (M <= 64).  Same arguments and outputs as analysis_batched;
    info[b] = iterations taken."""
    lib = load()
    for t, n in ((Yb, "Yb"), (d, "d"), (rinv_loc, "rinv_loc"), (Xb, "Xb")):
        _dev_f64(t, n)
    batch, p, M = Yb.shape
    nstate = Xb.shape[1]
    if d.shape != (batch, p) or rinv_loc.shape != (batch, p) or Xb.shape != (batch, nstate, M):
        raise LetkfError("inconsistent shapes")
    dev = Xb.device
    if Xa is None:
        Xa = torch.empty_like(Xb)
    W = torch.empty((batch, M, M), dtype=torch.float64, device=dev) if want_W else None
    wbar = torch.empty((batch, M), dtype=torch.float64, device=dev) if want_wbar else None
    if info is None:
        info = torch.zeros((batch,), dtype=torch.int32, device=dev)
    _out(Xa, "Xa", (batch, nstate, M), dev)
    _out(info, "info", (batch,), dev, torch.int32)
    with torch.cuda.device(dev):
        st = lib.letkf_analysis_batched_evdfree(_ptr(Yb), _ptr(d), _ptr(rinv_loc), _ptr(Xb), M, p, nstate, batch, float(rho),
                                                _ptr(Xa), _ptr(W), _ptr(wbar), _ptr(info), _stream(stream))
    _check(st, "letkf_analysis_batched_evdfree")
    return dict(Xa=Xa, W=W, wbar=wbar, info=info)


def analysis_grid(Yf, yo, Xb, hw, loc_kind, loc_scale, sigma_o, rho, obs_mask=None, Xa=None,
                  want_wbar=False, info=None, work=None, stream=None):
    """letkf_analysis_grid: Yf[V][Ny][Nx][M], yo[V][Ny][Nx], Xb[Ny*Nx][nstate][M] (device tensors)
    -> dict(Xa, wbar, info).  The local observations are gathered inside the library."""
    lib = load()
    _dev_f64(Yf, "Yf")
    _dev_f64(yo, "yo")
    _dev_f64(Xb, "Xb")
    V, Ny, Nx, M = Yf.shape
    nstate = Xb.shape[1]
    if yo.shape != (V, Ny, Nx) or Xb.shape != (Ny * Nx, nstate, M):
        raise LetkfError("inconsistent shapes")
    if obs_mask is not None and (obs_mask.dtype != torch.uint8 or obs_mask.shape != (Ny, Nx)
                                 or not obs_mask.is_cuda or not obs_mask.is_contiguous()):
        raise LetkfError("obs_mask must be a contiguous uint8 CUDA tensor [Ny][Nx]")
    dev = Xb.device
    if Xa is None:
        Xa = torch.empty_like(Xb)
    wbar = torch.empty((Ny * Nx, M), dtype=torch.float64, device=dev) if want_wbar else None
    if info is None:
        info = torch.zeros((Ny * Nx,), dtype=torch.int32, device=dev)
    _out(Xa, "Xa", (Ny * Nx, nstate, M), dev)
    _out(info, "info", (Ny * Nx,), dev, torch.int32)
    wb = _work(work, dev, lib.letkf_analysis_grid_workspace_bytes(M, V, Ny, Nx, int(hw), nstate))
    with torch.cuda.device(dev):
        st = lib.letkf_analysis_grid(_ptr(Yf), _ptr(yo), _ptr(obs_mask), _ptr(Xb), M, V, Ny, Nx, nstate, int(hw),
                                     int(loc_kind), float(loc_scale), float(sigma_o), float(rho),
                                     _ptr(Xa), _ptr(wbar), _ptr(info), _ptr(work), wb, _stream(stream))
    _check(st, "letkf_analysis_grid")
    return dict(Xa=Xa, wbar=wbar, info=info)


def analysis_grid_workspace_bytes(M, V, Ny, Nx, hw, nstate):
    return load().letkf_analysis_grid_workspace_bytes(M, V, Ny, Nx, hw, nstate)


def _host_f64(t, name):
    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise LetkfError(f"{name} must be a contiguous float64 CPU tensor (pinned for full copy speed)")
    return t


def syev_batched_host(A, w=None, V=None, info=None):
    """letkf_syev_batched_host: the EVD on HOST tensors (pinned memory recommended).  The library
    pipelines H2D copy, kernels and D2H copy; the call blocks until w, V, info are on the host."""
    lib = load()
    _host_f64(A, "A")
    batch, M, M2 = A.shape
    if M != M2:
        raise LetkfError("A must be [batch][M][M]")
    pin = A.is_pinned()
    if w is None:
        w = torch.empty((batch, M), dtype=torch.float64, pin_memory=pin)
    if V is None:
        V = torch.empty((batch, M, M), dtype=torch.float64, pin_memory=pin)
    if info is None:
        info = torch.zeros((batch,), dtype=torch.int32, pin_memory=pin)
    _host_f64(w, "w")
    _host_f64(V, "V")
    st = lib.letkf_syev_batched_host(_ptr(A), M, batch, _ptr(w), _ptr(V), _ptr(info))
    _check(st, "letkf_syev_batched_host")
    return w, V, info


def analysis_batched_host(Yb, d, rinv_loc, Xb, rho, Xa=None, want_W=False, want_wbar=False, info=None):
    """letkf_analysis_batched_host: the fused analysis on HOST tensors; blocks until done."""
    lib = load()
    for t, n in ((Yb, "Yb"), (d, "d"), (rinv_loc, "rinv_loc"), (Xb, "Xb")):
        _host_f64(t, n)
    batch, nstate, M = Xb.shape
    p = Yb.shape[1]
    if Yb.shape != (batch, p, M) or d.shape != (batch, p) or rinv_loc.shape != (batch, p):
        raise LetkfError("shape mismatch: Yb[batch][p][M], d[batch][p], rinv_loc[batch][p], Xb[batch][nstate][M]")
    pin = Xb.is_pinned()
    if Xa is None:
        Xa = torch.empty_like(Xb, pin_memory=pin)
    W = torch.empty((batch, M, M), dtype=torch.float64, pin_memory=pin) if want_W else None
    wbar = torch.empty((batch, M), dtype=torch.float64, pin_memory=pin) if want_wbar else None
    if info is None:
        info = torch.zeros((batch,), dtype=torch.int32, pin_memory=pin)
    st = lib.letkf_analysis_batched_host(_ptr(Yb), _ptr(d), _ptr(rinv_loc), _ptr(Xb), M, p, nstate, batch,
                                         float(rho), _ptr(Xa), _ptr(W), _ptr(wbar), _ptr(info))
    _check(st, "letkf_analysis_batched_host")
    return {"Xa": Xa, "W": W, "wbar": wbar, "info": info}


def analysis_grid_host(Yf, yo, Xb, hw, loc_kind, loc_scale, sigma_o, rho, obs_mask=None, Xa=None, want_wbar=False):
    """letkf_analysis_grid_host: the grid form on HOST tensors (pinned recommended); blocks until done."""
    lib = load()
    for t, n in ((Yf, "Yf"), (yo, "yo"), (Xb, "Xb")):
        _host_f64(t, n)
    V, Ny, Nx, M = Yf.shape
    nstate = Xb.shape[1]
    if yo.shape != (V, Ny, Nx) or Xb.shape != (Ny * Nx, nstate, M):
        raise LetkfError("inconsistent shapes")
    if obs_mask is not None and (obs_mask.dtype != torch.uint8 or obs_mask.shape != (Ny, Nx) or obs_mask.is_cuda
                                 or not obs_mask.is_contiguous()):
        raise LetkfError("obs_mask must be a contiguous uint8 CPU tensor [Ny][Nx]")
    pin = Xb.is_pinned()
    if Xa is None:
        Xa = torch.empty_like(Xb, pin_memory=pin)
    wbar = torch.empty((Ny * Nx, M), dtype=torch.float64, pin_memory=pin) if want_wbar else None
    info = torch.zeros((Ny * Nx,), dtype=torch.int32, pin_memory=pin)
    st = lib.letkf_analysis_grid_host(_ptr(Yf), _ptr(yo), _ptr(obs_mask), _ptr(Xb), M, V, Ny, Nx, nstate, int(hw),
                                      int(loc_kind), float(loc_scale), float(sigma_o), float(rho),
                                      _ptr(Xa), _ptr(wbar), _ptr(info))
    _check(st, "letkf_analysis_grid_host")
    return dict(Xa=Xa, wbar=wbar, info=info)


def host_release():
    load().letkf_host_release()


def probe_dfma(blocks, threads, iters, stream=None):
    """Launch the fp64-FMA throughput probe once; returns the number of FMAs it executes."""
    lib = load()
    sink = torch.empty((blocks * threads,), dtype=torch.float64, device="cuda")
    n = ctypes.c_ulonglong(0)
    st = lib.letkf_probe_dfma(_ptr(sink), blocks, threads, iters, ctypes.byref(n), _stream(stream))
    _check(st, "letkf_probe_dfma")
    return n.value, sink


def profile_enable(on):
    """0/False off; 1/True each kernel timed alone (one chunk, caller's stream); 2 timeline of the pipeline."""
    return load().letkf_profile_enable(int(on))


def profile_timeline():
    """[(kernel name, start ms relative to the first record, duration ms)] of the last compute call."""
    lib = load()
    out = []
    for i, (name, ms) in enumerate(profile_records()):
        t0 = ctypes.c_float()
        _check(lib.letkf_profile_record_start(i, ctypes.byref(t0)), "letkf_profile_record_start")
        out.append((name, t0.value, ms))
    return out


def profile_records():
    """[(kernel name, milliseconds)] of the last compute call (synchronises)."""
    lib = load()
    out = []
    for i in range(lib.letkf_profile_count()):
        name = ctypes.c_char_p()
        ms = ctypes.c_float()
        _check(lib.letkf_profile_record(i, ctypes.byref(name), ctypes.byref(ms)), "letkf_profile_record")
        out.append((name.value.decode(), ms.value))
    return out


def profile_rotations():
    return load().letkf_profile_rotations()


def profile_direct():
    return load().letkf_profile_direct()


def set_option(name, value):
    _check(load().letkf_set_option(name.encode(), int(value)), f"letkf_set_option({name})")

#!/usr/bin/env python
"""bench.py -- throughput of the LETKF hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Headline (BASELINE.json `metric`): batched fp64 syev matrices/s at M=64, batch 16384
(BASELINE config 3: A = ((M-1)/rho) I + Yb^T diag(r) Yb, p=98).  One step = one
letkf_syev_batched call over the whole batch.  The fused analysis (config 4) is timed as well and
reported under "analysis".  Prints ONE JSON line on rank 0.

--impl reference times the CPU oracle (oracle/, plain Jacobi) on the host cores on a bounded
sample of the same workload; it is a baseline, not a target.
"""
import argparse
import ctypes
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "batched fp64 syev matrices/s at M=64 (batch 16384); % of FP64/HBM roofline"
M_HEAD, BATCH_HEAD, P_HEAD = 64, 16384, 98
# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel per launch, from the one ncu --set full
# capture of this round (profiles/r02_ncu_key_metrics.txt names the command; ncu runs are never timed).  The
# capture launches the kernel on TRAFFIC_LAUNCH_MATRICES matrices; bench.py scales it to its own launch size.
NCU_DRAM_BYTES = {}          # filled from profiles/r02_traffic.txt when present ("kernel bytes matrices" per line)
SM_COUNT = 148
DFMA_PER_CLK_SM = 64          # fp64 FMA lanes per SM (4 SMSPs x 16), DESIGN.md section 6


def ncu_traffic(kernel, matrices):
    """dram bytes of one launch of `kernel` over `matrices` matrices, scaled from the committed ncu capture."""
    path = os.path.join(ROOT, "profiles", "r02_traffic.txt")
    try:
        for line in open(path):
            f = line.split()
            if len(f) >= 3 and not line.startswith("#") and f[0] == kernel:
                return float(f[1]) * matrices / float(f[2])
    except OSError:
        pass
    return None


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def syev_model_flops(M):
    return 9.0 * M ** 3                      # SURVEY.md section 8(d) convention


def syev_bytes(M):
    return 16.0 * M * M + 8.0 * M            # read A once, write V and w once


def analysis_model_flops(M, p, ns):
    return 2.0 * p * M * M + 2.0 * p * M + 9.0 * M ** 3 + 4.0 * M * M + 2.0 * M ** 3 + 2.0 * ns * M * M + M * M


def analysis_bytes(M, p, ns):
    return 8.0 * (p * M + 2 * p + 2 * ns * M)


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clock / throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        self.samples, self.reasons, self.stop_flag = [], set(), False
        self.max_mhz, self.power = None, []
        self.thread = None
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "hw_power_brake": getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            time.sleep(0.02)

    def start(self):
        if self.nv is not None:
            self.stop_flag = False
            self.thread = threading.Thread(target=self._loop, daemon=True)
            self.thread.start()

    def stop(self):
        self.stop_flag = True
        if self.thread is not None:
            self.thread.join()
        out = {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
               "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
               "samples": len(self.samples)}
        if self.power:
            out["power_w_max"] = round(max(self.power), 1)
        return out


# ------------------------------------------------------------------------------------------------
def time_oracle_syev(A, nthreads=0):
    import oracle
    oracle.build()
    t0 = time.perf_counter()
    _, _, info, nt = oracle.syev_batched(A, nthreads=nthreads)
    dt = time.perf_counter() - t0
    return A.shape[0] / dt, nt, dt


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from harness import workloads as wl
    sample = 4096
    A = wl.letkf_shaped(sample, M_HEAD, P_HEAD, config_index=3)
    for _ in range(args.warmup):
        time_oracle_syev(A[:64])
    t0 = time.perf_counter()
    nt = 0
    for _ in range(args.steps):
        _, nt, _ = time_oracle_syev(A)
    dt = time.perf_counter() - t0
    value = sample * args.steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "matrices/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "config3: syev fp64 M=64 LETKF-shaped p=98 (bounded sample of the 16384 batch)"},
        "cpu_baseline": {"value": value, "unit": "matrices/s", "cores": nt, "kind": "oracle",
                         "sample": f"first {sample} matrices of config 3 per step (cyclic Jacobi, OpenMP over the batch)"},
        "e2e": {"value": value, "unit": "matrices/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
def cusolver_compare(A_dev, steps=2):
    """cusolverDnDsyevjBatched on the same device matrices: comparison only, never in the product."""
    import torch
    lib = None
    for name in ("libcusolver.so.11", "libcusolver.so.12", "libcusolver.so"):
        for d in ("", os.path.join(os.path.dirname(torch.__file__), "lib") + "/", "/usr/local/cuda/lib64/"):
            try:
                lib = ctypes.CDLL(d + name)
                break
            except OSError:
                continue
        if lib is not None:
            break
    if lib is None:
        import glob
        cands = glob.glob(os.path.join(sys.prefix, "lib", "python*", "site-packages", "nvidia", "cusolver", "lib", "libcusolver.so*"))
        if not cands:
            return {"unavailable": "libcusolver not found"}
        lib = ctypes.CDLL(cands[0])
    batch, M, _ = A_dev.shape
    vp, ci = ctypes.c_void_p, ctypes.c_int
    h = vp()
    if lib.cusolverDnCreate(ctypes.byref(h)) != 0:
        return {"unavailable": "cusolverDnCreate failed"}
    lib.cusolverDnSetStream(h, vp(torch.cuda.current_stream().cuda_stream))
    params = vp()
    lib.cusolverDnCreateSyevjInfo(ctypes.byref(params))
    jobz, uplo = 1, 0            # CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER
    Awork = A_dev.clone()
    W = torch.empty((batch, M), dtype=torch.float64, device="cuda")
    info = torch.zeros((batch,), dtype=torch.int32, device="cuda")
    lwork = ci(0)
    lib.cusolverDnDsyevjBatched_bufferSize.argtypes = [vp, ci, ci, ci, vp, ci, vp, ctypes.POINTER(ci), vp, ci]
    st = lib.cusolverDnDsyevjBatched_bufferSize(h, jobz, uplo, M, vp(Awork.data_ptr()), M, vp(W.data_ptr()),
                                                ctypes.byref(lwork), params, batch)
    if st != 0:
        return {"unavailable": f"bufferSize status {st}"}
    work = torch.empty((max(lwork.value, 1),), dtype=torch.float64, device="cuda")
    lib.cusolverDnDsyevjBatched.argtypes = [vp, ci, ci, ci, vp, ci, vp, vp, ci, vp, vp, ci]
    times = []
    for it in range(steps + 1):
        Awork.copy_(A_dev)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        st = lib.cusolverDnDsyevjBatched(h, jobz, uplo, M, vp(Awork.data_ptr()), M, vp(W.data_ptr()),
                                         vp(work.data_ptr()), lwork.value, vp(info.data_ptr()), params, batch)
        e1.record()
        torch.cuda.synchronize()
        if st != 0:
            return {"unavailable": f"syevjBatched status {st}"}
        if it > 0:
            times.append(e0.elapsed_time(e1))
    # residual of its answer on a sample (column-major output == V^T in our row-major view)
    n = min(batch, 512)
    V = Awork[:n].transpose(1, 2)
    R = torch.matmul(A_dev[:n], V) - V * W[:n].unsqueeze(1)
    res = float((R.flatten(1).norm(dim=1) / A_dev[:n].flatten(1).norm(dim=1)).max())
    lib.cusolverDnDestroySyevjInfo(params)
    lib.cusolverDnDestroy(h)
    ms = float(np.median(times))
    return {"routine": "cusolverDnDsyevjBatched (default tol/sweeps)", "ms": ms,
            "matrices_per_s": batch / (ms * 1e-3), "max_residual_sample": res,
            "info_nonzero": int((info != 0).sum())}


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2308_03310_b200 import build as b, letkf, sharding
    from harness import workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); "
                         "use --impl reference for the CPU oracle baseline")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        b.build()
    if world > 1:
        dist.barrier()
    letkf.load()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        return sharding.max_over_ranks(x, device="cuda")

    M, B, p = M_HEAD, BATCH_HEAD, P_HEAD
    # weak scaling: every rank owns a full config-3 batch (its own seed); no data-path collective
    A_host = wl.letkf_shaped(B, M, p, config_index=3 + 1000 * rank)
    A = torch.from_numpy(A_host).cuda()
    w = torch.empty((B, M), dtype=torch.float64, device="cuda")
    V = torch.empty_like(A)
    info = torch.zeros((B,), dtype=torch.int32, device="cuda")
    work = torch.empty(letkf.syev_workspace_bytes(M, B), dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def step():
        letkf.syev_batched(A, w=w, V=V, info=info, work=work, stream=stream)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    assert int(info.abs().max()) == 0, "QL did not converge on the bench workload"
    if args.timeline:
        # one pipelined step with CUDA events around every kernel on the private stream it runs on
        # (letkf_profile_enable(2)): the evidence that QL overlaps the other two kernels
        letkf.profile_enable(2)
        step()
        torch.cuda.synchronize()
        if rank == 0:
            print("# kernel, start ms (relative to the first launch), duration ms, end ms")
            for name, t0, ms in letkf.profile_timeline():
                print(f"{name:28s} {t0:8.3f} {ms:8.3f} {t0 + ms:8.3f}")
        letkf.profile_enable(0)
        if world > 1:
            dist.destroy_process_group()
        return
    launches_per_step = letkf.last_launch_count()

    # ---- timed region: K steps as a user runs them (sub-chunk pipeline on), CUDA events on the
    # launching stream (the library joins its private streams back into it before returning)
    sampler = ClockSampler(local)
    kern = {}
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.start()
    e0.record(stream)
    recs_all = []
    for _ in range(args.steps):
        step()
        recs_all.append(None)
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    ms_step = ms_total / args.steps
    # per-kernel durations: 3 more steps with letkf_profile_enable(1) -- chunk after chunk on the caller's
    # stream with a workspace that holds the whole batch, i.e. ONE launch per kernel, each timed alone by
    # CUDA events on that stream
    work_all = torch.empty(letkf.syev_workspace_bytes(M, 1) * B, dtype=torch.uint8, device="cuda")
    letkf.profile_enable(True)
    nprof = 3
    rot_total = direct_total = 0
    nlaunch = {}
    for _ in range(nprof):
        letkf.syev_batched(A, w=w, V=V, info=info, work=work_all, stream=stream)
        for name, ms in letkf.profile_records():
            kern.setdefault(name, []).append(ms)
            nlaunch[name] = nlaunch.get(name, 0) + 1
        rot_total = letkf.profile_rotations()
        direct_total = letkf.profile_direct()
    letkf.profile_enable(False)
    del work_all
    kern_ms = {k: float(np.sum(v) / nprof) for k, v in kern.items()}
    launches_alone = {k: v // nprof for k, v in nlaunch.items()}
    rot_per_matrix = rot_total / float(B)
    direct_frac = direct_total / float(B)
    value = world * B / (ms_step * 1e-3)

    # ---- roofline of the dominant kernel.  Flops per matrix, as the kernels do them:
    #   fast_tridiag   4/3 M^3                       Householder reduction (the reflectors are kept, no explicit Q);
    #                  48 < M <= 64: fast_tridiag_head 4/3 (M^3 - 32^3) + fast_tridiag_tail 4/3 32^3
    #   ql_log_kernel  30 flops per rotation step    (scalar recurrences; latency bound, not a roofline kernel)
    #   fast_apply     2 M^3 back-transform + 6 M R  (R logged rotations replayed) + 60 M^2 for a matrix whose
    #                  eigenvectors come from twisted factorisations (5 passes of ~12 flops per entry)
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak_derived = SM_COUNT * DFMA_PER_CLK_SM * 2 * sm_max * 1e6 / 1e12
    flops_per_matrix = {}
    split = any("tridiag_tail" in k for k in kern_ms)           # the reduction as two kernels: pivots M-1 ... 33, then 32 ... 1
    tail_flops = (4.0 / 3.0) * 32 ** 3
    for k in kern_ms:
        if "tridiag_tail" in k:
            flops_per_matrix[k] = tail_flops
        elif "tridiag" in k:
            flops_per_matrix[k] = (4.0 / 3.0) * M ** 3 - (tail_flops if split else 0.0)
        elif "apply" in k:
            flops_per_matrix[k] = 2.0 * M ** 3 + 6.0 * M * rot_per_matrix + 60.0 * M * M * direct_frac
        elif "ql" in k:
            flops_per_matrix[k] = 30.0 * 1.05 * M * M
    dom = max(kern_ms, key=kern_ms.get)
    dom_flops = flops_per_matrix.get(dom, 0.0) * B
    achieved = dom_flops / (kern_ms[dom] * 1e-3) / 1e12
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = peaks.get("hbm_gbs", 6650.0)

    # the fp64 peak, measured in this run: MEASURED_PEAKS.json has no fp64 entry and the profiling guide no
    # fp64 nominal, so the roofline denominator is the library's own DFMA probe (8 independent FMA chains per
    # thread, 8 CTAs of 256 threads per SM), timed here with CUDA events
    nfma, _ = letkf.probe_dfma(SM_COUNT * 8, 256, 2048)
    torch.cuda.synchronize()
    best = 0.0
    for _ in range(3):
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        p0.record(stream)
        nfma, _ = letkf.probe_dfma(SM_COUNT * 8, 256, 2048)
        p1.record(stream)
        torch.cuda.synchronize()
        best = max(best, 2.0 * nfma / (p0.elapsed_time(p1) * 1e-3) / 1e12)
    peak_measured = best

    algorithmic_bytes = {"fast_tridiag": (8.0 * M * M + 8.0 * (M * M / 2 + 3 * M)) * B,        # A in; reflectors, d, e out
                         # head: A in; reflectors of pivots >= 33, their (d, e), the 640-entry hand-over record out
                         "fast_tridiag_head": (8.0 * M * M + 8.0 * (M * M / 2 - 528 + 3 * (M - 32) + 640)) * B,
                         "fast_tridiag_tail": (8.0 * 640 + 8.0 * (528 + 3 * 32)) * B,          # hand-over in; the rest out
                         "ql_log_kernel": (16.0 * M + 12.0 * M + 16.0 * rot_per_matrix) * B,
                         "fast_apply": (8.0 * (M * M / 2 + 4 * M) + 16.0 * rot_per_matrix + 8.0 * M * M) * B}
    step_tflops = syev_model_flops(M) * B / (ms_step * 1e-3) / 1e12
    counted = (4.0 / 3.0) * M ** 3 + 2.0 * M ** 3 + 6.0 * M * rot_per_matrix + 60.0 * M * M * direct_frac
    roofline = {
        "bound": "alu", "kernel": dom, "achieved": achieved, "peak": peak_measured, "unit": "TFLOP/s",
        "frac": achieved / peak_measured,
        "peak_source": "measured in this run: letkf_probe_dfma (fp64 FMA, 148 x 8 CTAs x 256 threads x 8 chains), CUDA events",
        "peak_derived": peak_derived,
        "peak_derived_source": f"{SM_COUNT} SMs x {DFMA_PER_CLK_SM} DFMA/clk x 2 x {sm_max:.0f} MHz (DESIGN.md 5)",
        "frac_of_derived": achieved / peak_derived,
        "flops_per_launch": dom_flops, "matrices_per_launch": B, "launches_timed_alone": launches_alone.get(dom),
        "traffic": ncu_traffic(dom, B),
        "traffic_unit": "bytes per launch (whole batch): ncu dram read+write of profiles/r02_traffic.txt scaled to this launch; null = no capture committed",
        "algorithmic_bytes": algorithmic_bytes.get(dom),
        "kernel_ms": kern_ms, "kernel_share": {k: v / sum(kern_ms.values()) for k, v in kern_ms.items()},
        "kernel_flops_per_matrix": flops_per_matrix,
        "kernel_frac_of_measured_peak": {k: flops_per_matrix[k] * B / (kern_ms[k] * 1e-3) / 1e12 / peak_measured
                                         for k in kern_ms if k in flops_per_matrix},
        "rotations_per_matrix": rot_per_matrix, "direct_eigenvector_fraction": direct_frac,
        "flops_counted_per_matrix": counted,
        "step_counted": {"achieved": counted * B / (ms_step * 1e-3) / 1e12,
                         "frac_of_measured": counted * B / (ms_step * 1e-3) / 1e12 / peak_measured},
        "step_model_9M3": {"achieved": step_tflops, "frac_of_measured": step_tflops / peak_measured,
                           "frac_of_derived": step_tflops / peak_derived,
                           "note": "9 M^3 is SURVEY.md 8(d)'s textbook model of Householder + QL with accumulated rotations + back-transform; "
                                   "the path does flops_counted_per_matrix (no rotation is applied where the eigenvectors of T are formed directly)"},
        "step_hbm": {"achieved_gbs": syev_bytes(M) * B / (ms_step * 1e-3) / 1e9,
                     "peak_gbs": hbm_peak, "frac": syev_bytes(M) * B / (ms_step * 1e-3) / 1e9 / hbm_peak},
        "workspace_bytes": int(work.numel()),
    }

    # ---- end to end through the C ABI with HOST buffers (letkf_syev_batched_host): pinned inputs
    # and outputs, the library's own chunked H2D -> kernels -> D2H pipeline inside the timed region
    A_pin = torch.from_numpy(A_host).pin_memory()
    w_pin = torch.empty((B, M), dtype=torch.float64).pin_memory()
    V_pin = torch.empty((B, M, M), dtype=torch.float64).pin_memory()
    i_pin = torch.zeros((B,), dtype=torch.int32).pin_memory()

    def e2e_step():
        letkf.syev_batched_host(A_pin, w=w_pin, V=V_pin, info=i_pin)      # blocks until V_pin is written

    e2e_step()
    e2e_launches = letkf.last_launch_count()
    barrier()
    ksteps = min(args.steps, 5)
    e0.record(stream)
    for _ in range(ksteps):
        e2e_step()
    e1.record(stream)
    barrier()
    e2e_ms = max_over_ranks(e0.elapsed_time(e1)) / ksteps
    assert int(i_pin.abs().max()) == 0 and torch.equal(w_pin, w.cpu()), "e2e result differs from the device call"
    e2e = {"value": world * B / (e2e_ms * 1e-3), "unit": "matrices/s",
           "h2d_bytes_per_step": int(A_pin.numel() * 8),
           "d2h_bytes_per_step": int((w_pin.numel() + V_pin.numel()) * 8 + i_pin.numel() * 4),
           "ms_per_step": e2e_ms, "steps": ksteps, "gpu_launches_per_step": e2e_launches,
           "api": "letkf_syev_batched_host, pinned host buffers"}
    del A_pin, V_pin
    letkf.host_release()

    line = {
        "metric": METRIC, "value": value, "unit": "matrices/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "config3: letkf_syev_batched fp64 M=64 batch=16384 per GPU, LETKF-shaped p=98 rho=1.1",
                   "l2": "inputs larger than L2: A+V = 1 GiB per step, no flush needed"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * args.steps,
        "roofline": roofline,
    }

    if rank == 0 and world == 1:
        # ---- fused analysis (config 4), same protocol
        if not args.no_analysis:
            inp = wl.analysis_inputs()
            t = {k: torch.from_numpy(inp[k]).cuda() for k in ("Yb", "d", "rinv_loc", "Xb")}
            Xa = torch.empty_like(t["Xb"])
            awork = torch.empty(letkf.analysis_workspace_bytes(M, p, 9, B), dtype=torch.uint8, device="cuda")

            def astep():
                letkf.analysis_batched(t["Yb"], t["d"], t["rinv_loc"], t["Xb"], inp["rho"], Xa=Xa, info=info,
                                       work=awork, stream=stream)
            for _ in range(3):
                astep()
            torch.cuda.synchronize()
            e0.record(stream)
            for _ in range(args.steps):
                astep()
            e1.record(stream)
            torch.cuda.synchronize()
            ams = e0.elapsed_time(e1) / args.steps
            fl = analysis_model_flops(M, p, 9)
            line["analysis"] = {
                "workload": "config4: letkf_analysis_batched fp64 M=64 p=98 nstate=9, 128x128 grid points, W not requested",
                "value": B / (ams * 1e-3), "unit": "grid points/s", "ms_per_step": ams,
                "gpu_launches_per_step": letkf.last_launch_count(),
                "model_tflops": fl * B / (ams * 1e-3) / 1e12, "frac_of_measured_fp64_peak": fl * B / (ams * 1e-3) / 1e12 / peak_measured,
                "workspace_bytes": int(awork.numel()),
                "hbm_gbs": analysis_bytes(M, p, 9) * B / (ams * 1e-3) / 1e9}
            letkf.profile_enable(True)
            astep()
            akern = {}
            for k, v in letkf.profile_records():
                akern[k] = akern.get(k, 0.0) + v
            line["analysis"]["kernel_ms"] = {k: round(v, 4) for k, v in akern.items()}
            line["analysis"]["direct_eigenvector_fraction"] = letkf.profile_direct() / float(B)
            letkf.profile_enable(False)
            # the EVD-free form of the same analysis: coupled Newton-Schulz on the FP64 tensor cores
            ninfo = torch.zeros((B,), dtype=torch.int32, device="cuda")
            nXa = torch.empty_like(t["Xb"])
            for _ in range(2):
                letkf.analysis_batched_evdfree(t["Yb"], t["d"], t["rinv_loc"], t["Xb"], inp["rho"], Xa=nXa, info=ninfo, stream=stream)
            torch.cuda.synchronize()
            e0.record(stream)
            for _ in range(min(args.steps, 5)):
                letkf.analysis_batched_evdfree(t["Yb"], t["d"], t["rinv_loc"], t["Xb"], inp["rho"], Xa=nXa, info=ninfo, stream=stream)
            e1.record(stream)
            torch.cuda.synchronize()
            nms = e0.elapsed_time(e1) / min(args.steps, 5)
            nit = float(ninfo.float().mean())
            line["analysis"]["evdfree"] = {
                "api": "letkf_analysis_batched_evdfree (coupled Newton-Schulz, mma.sync.m8n8k4.f64)", "ms_per_step": nms,
                "value": B / (nms * 1e-3), "unit": "grid points/s", "iterations_mean": nit,
                "dmma_tflops": (3 * nit * 2.0 * M ** 3 + 2.0 * p * M * M) * B / (nms * 1e-3) / 1e12,
                "max_rel_diff_Xa_vs_evd_route": float(((nXa - Xa).flatten(1).norm(dim=1) / (Xa - t["Xb"].mean(dim=2, keepdim=True)).flatten(1).norm(dim=1)).max())}
            del nXa, ninfo
            # end to end through letkf_analysis_batched_host (pinned host buffers, PCIe inside)
            hp = {k: torch.from_numpy(inp[k]).pin_memory() for k in ("Yb", "d", "rinv_loc", "Xb")}
            Xa_pin = torch.empty_like(hp["Xb"]).pin_memory()
            letkf.analysis_batched_host(hp["Yb"], hp["d"], hp["rinv_loc"], hp["Xb"], inp["rho"], Xa=Xa_pin)
            ksteps = min(args.steps, 3)
            e0.record(stream)
            for _ in range(ksteps):
                letkf.analysis_batched_host(hp["Yb"], hp["d"], hp["rinv_loc"], hp["Xb"], inp["rho"], Xa=Xa_pin)
            e1.record(stream)
            torch.cuda.synchronize()
            hms = e0.elapsed_time(e1) / ksteps
            assert torch.equal(Xa_pin, Xa.cpu()), "analysis e2e result differs from the device call"
            line["analysis"]["e2e"] = {
                "value": B / (hms * 1e-3), "unit": "grid points/s", "ms_per_step": hms,
                "h2d_bytes_per_step": int(sum(v.numel() for v in hp.values()) * 8),
                "d2h_bytes_per_step": int(Xa_pin.numel() * 8 + B * 4), "api": "letkf_analysis_batched_host"}
            del hp, Xa_pin
            letkf.host_release()
            # ---- the analysis above the register kernels (a1/a2 and a6-a9 are launches of their own there:
            # big_gram (FP64 tensor cores) -> EVD -> generic_epilogue), the sweep's batch sizes
            line["analysis_large"] = []
            for Ml in (128, 256):
                Bl = wl.sweep_batch(Ml)
                li = wl.analysis_inputs(batch=Bl, M=Ml, p=98, nstate=9, config_index=70)
                lt = {k: torch.from_numpy(li[k]).cuda() for k in ("Yb", "d", "rinv_loc", "Xb")}
                lXa = torch.empty_like(lt["Xb"])
                linfo = torch.zeros((Bl,), dtype=torch.int32, device="cuda")
                lwork = torch.empty(letkf.analysis_workspace_bytes(Ml, 98, 9, Bl), dtype=torch.uint8, device="cuda")
                for _ in range(2):
                    letkf.analysis_batched(lt["Yb"], lt["d"], lt["rinv_loc"], lt["Xb"], li["rho"], Xa=lXa, info=linfo, work=lwork, stream=stream)
                torch.cuda.synchronize()
                ks = min(args.steps, 5)
                e0.record(stream)
                for _ in range(ks):
                    letkf.analysis_batched(lt["Yb"], lt["d"], lt["rinv_loc"], lt["Xb"], li["rho"], Xa=lXa, info=linfo, work=lwork, stream=stream)
                e1.record(stream)
                torch.cuda.synchronize()
                lms = e0.elapsed_time(e1) / ks
                fl = analysis_model_flops(Ml, 98, 9)
                line["analysis_large"].append({
                    "workload": f"letkf_analysis_batched fp64 M={Ml} p=98 nstate=9 batch={Bl}, W not requested",
                    "ms_per_step": round(lms, 4), "value": Bl / (lms * 1e-3), "unit": "grid points/s",
                    "frac_of_measured_fp64_peak": round(fl * Bl / (lms * 1e-3) / 1e12 / peak_measured, 4),
                    "info_nonzero": int((linfo != 0).sum())})
                del lt, lXa, linfo, lwork
            # ---- grid form: same 128 x 128 x 2 x 7x7 problem, the local
            # observations gathered inside the library from the fields (Y_loc never materialised)
            gi = wl.grid_inputs()
            gt = {k: torch.from_numpy(gi[k]).cuda() for k in ("Yf", "yo", "Xb")}
            gXa = torch.empty_like(gt["Xb"])
            gwork = torch.empty(letkf.analysis_grid_workspace_bytes(M, 2, 128, 128, 3, 9), dtype=torch.uint8, device="cuda")

            def gstep():
                letkf.analysis_grid(gt["Yf"], gt["yo"], gt["Xb"], 3, 0, 2.0, gi["sigma_o"], gi["rho"], Xa=gXa,
                                    info=info, work=gwork, stream=stream)
            for _ in range(3):
                gstep()
            torch.cuda.synchronize()
            e0.record(stream)
            for _ in range(args.steps):
                gstep()
            e1.record(stream)
            torch.cuda.synchronize()
            gms = e0.elapsed_time(e1) / args.steps
            gl = letkf.last_launch_count()
            hp = {k: torch.from_numpy(gi[k]).pin_memory() for k in ("Yf", "yo", "Xb")}
            gXa_pin = torch.empty_like(hp["Xb"]).pin_memory()
            letkf.analysis_grid_host(hp["Yf"], hp["yo"], hp["Xb"], 3, 0, 2.0, gi["sigma_o"], gi["rho"], Xa=gXa_pin)
            ksteps = min(args.steps, 3)
            e0.record(stream)
            for _ in range(ksteps):
                letkf.analysis_grid_host(hp["Yf"], hp["yo"], hp["Xb"], 3, 0, 2.0, gi["sigma_o"], gi["rho"], Xa=gXa_pin)
            e1.record(stream)
            torch.cuda.synchronize()
            ghms = e0.elapsed_time(e1) / ksteps
            assert torch.equal(gXa_pin, gXa.cpu()), "grid e2e result differs from the device call"
            line["analysis_grid"] = {
                "workload": "letkf_analysis_grid fp64 M=64 V=2 128x128 periodic grid, 7x7 patch (p=98), nstate=9, Gaussian localisation",
                "value": B / (gms * 1e-3), "unit": "grid points/s", "ms_per_step": gms, "gpu_launches_per_step": gl,
                "hbm_bytes_per_point_algorithmic": 8.0 * (2 * 65 + 2 * 9 * M),
                "e2e": {"value": B / (ghms * 1e-3), "unit": "grid points/s", "ms_per_step": ghms,
                        "h2d_bytes_per_step": int(sum(v.numel() for v in hp.values()) * 8),
                        "d2h_bytes_per_step": int(gXa_pin.numel() * 8 + B * 4), "api": "letkf_analysis_grid_host"}}
            del gi, gt, gXa, gwork, hp, gXa_pin
            letkf.host_release()
            del t, Xa, awork, inp
        # ---- config 5: EVD size sweep, batch = floor(2^26 / M^2), LETKF-shaped
        if not args.no_sweep:
            sweep = []
            del A, V, w, work
            torch.cuda.empty_cache()
            for Ms in (16, 32, 48, 64, 96, 128, 192, 256):
                Bs = (1 << 26) // (Ms * Ms)
                As = torch.from_numpy(wl.config5(Ms, batch=Bs)).cuda()
                ws_ = torch.empty((Bs, Ms), dtype=torch.float64, device="cuda")
                Vs = torch.empty_like(As)
                infos = torch.zeros((Bs,), dtype=torch.int32, device="cuda")
                wk = torch.empty(letkf.syev_workspace_bytes(Ms, Bs), dtype=torch.uint8, device="cuda")
                for _ in range(3):
                    letkf.syev_batched(As, w=ws_, V=Vs, info=infos, work=wk, stream=stream)
                torch.cuda.synchronize()
                nrep = 3
                e0.record(stream)
                for _ in range(nrep):
                    letkf.syev_batched(As, w=ws_, V=Vs, info=infos, work=wk, stream=stream)
                e1.record(stream)
                torch.cuda.synchronize()
                sms = e0.elapsed_time(e1) / nrep
                tf = syev_model_flops(Ms) * Bs / (sms * 1e-3) / 1e12
                sweep.append({"M": Ms, "batch": Bs, "ms": round(sms, 4), "matrices_per_s": Bs / (sms * 1e-3),
                              "model_9M3_tflops": round(tf, 3), "frac_of_measured_fp64_peak": round(tf / peak_measured, 4),
                              "workspace_bytes": int(wk.numel()),
                              "path": "registers (fast_*)" if Ms <= 64 else ("registers + shared memory (mid_*)" if Ms <= 160 else "global/L2 (generic_*)"),
                              "info_nonzero": int((infos != 0).sum())})
                del As, Vs, ws_, wk, infos
            line["sweep"] = sweep
            # the paper's Table I shapes (batch 16384 at M = 16, 32, 48, 64, A100 FP32:
            # 1.3 / 2.4 / 7.8 / 14.2 ms) and its 64-GPU share of 256 matrices per GPU
            shapes = []
            for Ms, ps in ((16, 49), (32, 49), (48, 49), (64, 98)):
                for Bs in (16384, 256):
                    As = torch.from_numpy(wl.letkf_shaped(Bs, Ms, ps, config_index=80 + Ms)).cuda()
                    ws_ = torch.empty((Bs, Ms), dtype=torch.float64, device="cuda")
                    Vs = torch.empty_like(As)
                    wk = torch.empty(letkf.syev_workspace_bytes(Ms, Bs), dtype=torch.uint8, device="cuda")
                    for _ in range(3):
                        letkf.syev_batched(As, w=ws_, V=Vs, work=wk, stream=stream)
                    torch.cuda.synchronize()
                    e0.record(stream)
                    for _ in range(10):
                        letkf.syev_batched(As, w=ws_, V=Vs, work=wk, stream=stream)
                    e1.record(stream)
                    torch.cuda.synchronize()
                    sms = e0.elapsed_time(e1) / 10
                    shapes.append({"M": Ms, "batch": Bs, "ms": round(sms, 4), "matrices_per_s": Bs / (sms * 1e-3)})
                    del As, Vs, ws_, wk
            line["paper_shapes_fp64"] = shapes
            # the same shapes in the paper's precision (letkf_syev_batched_f32); the
            # paper's own numbers are FP32 on one A100 (context, another machine)
            paper_ms = {16: 1.3, 32: 2.4, 48: 7.8, 64: 14.2}
            shapes32 = []
            for Ms, ps in ((16, 49), (32, 49), (48, 49), (64, 98)):
                Bs = 16384
                As = torch.from_numpy(wl.letkf_shaped(Bs, Ms, ps, config_index=80 + Ms).astype(np.float32)).cuda()
                ws_ = torch.empty((Bs, Ms), dtype=torch.float32, device="cuda")
                Vs = torch.empty_like(As)
                wk = torch.empty(letkf.syev_f32_workspace_bytes(Ms, Bs), dtype=torch.uint8, device="cuda")
                for _ in range(3):
                    letkf.syev_batched_f32(As, w=ws_, V=Vs, work=wk, stream=stream)
                torch.cuda.synchronize()
                e0.record(stream)
                for _ in range(10):
                    letkf.syev_batched_f32(As, w=ws_, V=Vs, work=wk, stream=stream)
                e1.record(stream)
                torch.cuda.synchronize()
                sms = e0.elapsed_time(e1) / 10
                shapes32.append({"M": Ms, "batch": Bs, "ms": round(sms, 4), "matrices_per_s": Bs / (sms * 1e-3),
                                 "paper_a100_fp32_ms": paper_ms[Ms]})
                del As, Vs, ws_, wk
            line["paper_shapes_fp32"] = shapes32
            A = torch.from_numpy(A_host).cuda()
        # ---- cuSOLVER on the same matrices (comparison only)
        if not args.no_cusolver:
            try:
                line["cusolver"] = cusolver_compare(A)
            except Exception as ex:          # comparison must never break the bench
                line["cusolver"] = {"unavailable": repr(ex)[:200]}
        # ---- CPU baseline: the oracle on the host cores, bounded sample
        if not args.no_cpu_baseline:
            sample = 8192
            v, nt, dt = time_oracle_syev(A_host[:sample])
            line["cpu_baseline"] = {"value": v, "unit": "matrices/s", "cores": nt, "kind": "oracle",
                                    "sample": f"first {sample} matrices of config 3 (cyclic Jacobi fp64, OpenMP over the batch), {dt:.1f} s"}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-analysis", action="store_true")
    ap.add_argument("--no-cusolver", action="store_true")
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--timeline", action="store_true", help="print the kernel timeline of one pipelined step and exit")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

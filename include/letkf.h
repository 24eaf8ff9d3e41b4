/*
 * letkf.h -- C ABI of libletkf: the per-grid-point LETKF local analysis of
 * arXiv 2308.03310 (Hasegawa et al., "GPU Optimization of Lattice Boltzmann Method with
 * Local Ensemble Transform Kalman Filter"), hand-written CUDA for sm_100a (NVIDIA B200).
 *
 * Citations are "PAPER.md:<line>" of the paper text plus the equation / section.
 *
 * General contract (every entry point):
 *   - every array pointer is a DEVICE pointer owned by the caller (for instance the data_ptr
 *     of a torch tensor).  Arrays are row-major, batch outermost ("the batch
 *     dimension is the outermost"), fp64, 16-byte aligned.
 *   - work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = legacy default
 *     stream) and the call returns without synchronising.  Internally the library may fork
 *     onto private streams that are joined back into `stream` before the call returns, so
 *     stream order is all a caller needs.
 *   - workspace: `work` is a caller-owned device buffer; the matching letkf_*_workspace_bytes()
 *     returns the RECOMMENDED size (all sub-chunks of the call in flight).  Any size that holds one
 *     matrix's records is accepted -- the call then keeps fewer sub-chunks in flight or runs chunk
 *     after chunk -- and a smaller one is refused (-k).  If `work` is NULL the library takes it from
 *     the device's default memory pool with cudaMallocAsync / cudaFreeAsync on `stream`
 *     (stream-ordered, no synchronisation).
 *   - return value: 0 = LETKF_OK; -k = the k-th argument (1-based) is invalid (NULL where
 *     not allowed, out of range, misaligned); >0 = a cudaError_t from the launch.
 *     Per-matrix numerical status is asynchronous, in info[b] (see below).
 *   - inputs are never written unless aliased with an output as documented.
 *   - there is NO CPU fallback: without a CUDA device every compute call returns a
 *     cudaError_t.
 *   - results are bitwise reproducible run to run for fixed inputs (no floating-point atomics).
 */
#ifndef LETKF_H
#define LETKF_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LETKF_OK 0
#define LETKF_MAX_M 256       /* largest ensemble size / matrix order accepted            */
#define LETKF_VERSION 100     /* major*10000 + minor*100 + patch                          */

/* info[b] bit flags (0 = converged on the fast path) */
#define LETKF_INFO_SLOWPATH 0x40000000 /* the matrix was finished by the in-kernel slow path
                                          (rotation log full, or a QL rotation with f^2 + g^2
                                          outside [1e-280, 1e280]); result is still valid   */
/* info[b] & 0xFFFF = number of off-diagonal elements that had not converged after 60
 * QL iterations each ("implicit QL method ... as in EISPACK/LAPACK"; twice the
 * cap of EISPACK tql2).  Non-zero means w/V of that matrix are not to be trusted.                */

/*
 * Batched symmetric eigenvalue decomposition -- the paper's "main computing kernel"
 * ("computed by the eigenvalue decomposition (EVD) of Q", section III
 * Householder tridiagonalisation -> implicit QL -> back-transform).
 *
 *   A[b] = V[b] diag(w[b]) V[b]^T,  V[b]^T V[b] = I,  w[b] ascending.
 *
 *   A     in   [batch][M][M]  symmetric; only the LOWER triangle (row >= col) is read.
 *   M          matrix order, 1 <= M <= LETKF_MAX_M
 *   batch      number of matrices, >= 0 (0 = successful no-op)
 *   w     out  [batch][M]     eigenvalues, ascending
 *   V     out  [batch][M][M]  eigenvector k is COLUMN k: A[b] @ V[b] == V[b] * w[b]
 *                             (numpy.linalg.eigh convention).  V may alias A (in place).
 *                             Sign of each eigenvector (and the basis inside a repeated
 *                             eigenvalue) is not specified.
 *   info  out  [batch] ints or NULL
 *   work       device workspace or NULL, work_bytes >= letkf_syev_workspace_bytes(M, batch)
 *   stream     cudaStream_t
 *
 * Precondition: entries finite with 1e-100 < max|A| < 1e100 (no rescaling is applied);
 * non-finite input terminates (iteration cap: 60 sweeps per eigenvalue) with info[b] != 0.
 */
int letkf_syev_batched(const double* A, int M, int batch, double* w, double* V,
                       int* info, void* work, size_t work_bytes, void* stream);

size_t letkf_syev_workspace_bytes(int M, int batch);

/*
 * letkf_syev_batched for callers that may not allocate (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): same arguments and results, but there is no
 * workspace argument and the call makes NO cudaMalloc / cudaFree / cudaMallocAsync, creates no
 * stream and no event.  The scratch memory of the kernels (reflectors, (d, e), rotation log, flags:
 * DESIGN.md section 4) is a file-scope `static __device__` array of LETKF_STATIC_WORK_BYTES inside the
 * library, which every GPU that loads the library holds until the process exits.  All kernels
 * (reduction, eigenvalues, apply) are launched one after the other on `stream`; the kernels and the
 * results are those of letkf_syev_batched at the same batch size.
 *
 *   batch   must fit the array: batch <= letkf_syev_static_max_batch(M) (paper's latency case, 256
 *           matrices of M = 64, fits; M = 64: 363, M = 32: 1297, M = 16: 4123, M = 128: 92, M = 256: 31), else
 *           the call returns LETKF_ERR_STATIC_CAPACITY and launches nothing.
 *   Every call on a device shares the one array: two calls whose kernels overlap on the GPU (different
 *   streams, or different host threads) RACE on it -- keep all calls of a device on one stream or order
 *   them with events.  The array keeps the last call's contents; the call clears the per-matrix flag
 *   and sweep-count records it starts from (every other record is written before it is read).
 *   Profiling records (letkf_profile_enable) are not taken by this entry point.
 */
#define LETKF_STATIC_WORK_BYTES (32u << 20)
#define LETKF_ERR_STATIC_CAPACITY (-100)
int letkf_syev_batched_static(const double* A, int M, int batch, double* w, double* V,
                              int* info, void* stream);

/* largest batch letkf_syev_batched_static accepts for order M (0 for an invalid M) */
int letkf_syev_static_max_batch(int M);

/*
 * The same decomposition in the paper's precision ("single-precision"; Table I,
 * M = 16, 32, 48, 64, batch 128^2): A, w, V are fp32.  SURVEY.md section 8(f) N2.
 * The Householder reduction, the replay of plane rotations and the back-transform run in fp32; the
 * tridiagonal eigenproblem (O(M^2) of the O(M^3) work) is solved in fp64 on the (d, e) the fp32
 * reduction produced, so the result is the EVD of a matrix within a few eps32 ||A|| of A:
 *   max_k |w_k - lambda_k| <~ 50 eps32 ||A||_2,  ||A V - V diag(w)||_F / ||A||_F <~ 100 eps32,
 *   max |V^T V - I| <~ 100 eps32                                   (eps32 = 2^-24)
 * 1 <= M <= 64 (the register-resident path); other arguments, info and the workspace as for
 * letkf_syev_batched (size from letkf_syev_f32_workspace_bytes).  V may alias A.
 */
int letkf_syev_batched_f32(const float* A, int M, int batch, float* w, float* V,
                           int* info, void* work, size_t work_bytes, void* stream);

size_t letkf_syev_f32_workspace_bytes(int M, int batch);

/*
 * Fused LETKF local analysis of `batch` grid points (Eq.13-19;
 * Procedure 1 lines 5-7).  For each point, with dY = Yb (p x M),
 * r = rinv_loc (the diagonal of G o R^-1), dvec = d = y^o - ybar^f:
 *
 *   Q     = ((M-1)/rho) I + dY^T diag(r) dY                        Eq.17 (rho = 1 is the paper's)
 *   Q     = V diag(lam) V^T
 *   wbar  = V diag(1/lam) V^T dY^T diag(r) dvec                    Eq.14, Eq.16
 *   W     = sqrt(M-1) V diag(lam^-1/2) V^T                         Eq.15, symmetric square root
 *   xbar  = mean_m Xb[:, m],  dX = Xb - xbar                       Eq.9-11
 *   Xa    = xbar 1^T + dX (wbar 1^T + W)                           Eq.13
 *
 *   Yb        in  [batch][p][M]       observation-space perturbations (rows centred by the caller)
 *   d         in  [batch][p]          innovations
 *   rinv_loc  in  [batch][p]          >= 0; 0 marks a padded / ignored observation
 *   Xb        in  [batch][nstate][M]  background ensemble (members, not perturbations)
 *   M, p, nstate, batch               2 <= M <= LETKF_MAX_M (one member has no spread), p >= 0, nstate >= 1, batch >= 0
 *   rho                               multiplicative covariance inflation, > 0
 *   Xa        out [batch][nstate][M]  analysis ensemble; may alias Xb
 *   W         out [batch][M][M] or NULL
 *   wbar      out [batch][M]    or NULL
 *   info      out [batch] or NULL     as for letkf_syev_batched
 *   work / work_bytes / stream        as above, size from letkf_analysis_workspace_bytes()
 */
int letkf_analysis_batched(const double* Yb, const double* d, const double* rinv_loc,
                           const double* Xb, int M, int p, int nstate, int batch, double rho,
                           double* Xa, double* W, double* wbar, int* info,
                           void* work, size_t work_bytes, void* stream);

size_t letkf_analysis_workspace_bytes(int M, int p, int nstate, int batch);

/*
 * The same analysis WITHOUT an eigendecomposition (the paper's stated
 * future work, "explore algorithms that can avoid divergence"): Eq.14-16 need only
 * Q^-1 applied to a vector and the symmetric square root Q^-1/2, and both come out of a coupled
 * Newton-Schulz iteration  T = (3I - Z Y)/2, Y <- Y T, Z <- Z T  started from Y = Q/c, Z = I
 * (Y -> (Q/c)^1/2, Z -> (Q/c)^-1/2; c from the trace bound of lambda_max and the known lower bound
 * (M-1)/rho of lambda_min).  Every step is a dense M x M x M product on the FP64 tensor cores
 * (mma.sync.m8n8k4.f64), no data-dependent branch but the convergence test ||I - Z Y||_F <=
 * 1e-14 sqrt(M) (or its rounding floor).  Same inputs and outputs as letkf_analysis_batched; W and Xa
 * agree with it to ~3e-14 kappa(Q)^2 relative (the coupled iteration is not backward stable): inside the
 * 1e-10 tolerance for kappa(Q) <~ 50 (config 4: kappa ~ 4, 1e-12; 3e-9 at kappa ~ 300, 2e-7 at 3e3).  Iterations ~ 4 + log_1.5 sqrt(kappa').
 * 2 <= M <= 64, nstate <= 16; no workspace.  info[b] = iterations taken, or
 * LETKF_INFO_NS_NOCONV | iterations if the tolerance was not reached in 40 (result not to be trusted).
 * Measured slower than the EVD route on B200 (fp64 tensor rate = vector rate).
 */
#define LETKF_INFO_NS_NOCONV 0x20000000
int letkf_analysis_batched_evdfree(const double* Yb, const double* d, const double* rinv_loc,
                                   const double* Xb, int M, int p, int nstate, int batch, double rho,
                                   double* Xa, double* W, double* wbar, int* info, void* stream);

/*
 * Grid form of the fused analysis (PAPER.md:144-151 R-localisation,
 * Procedure 1 lines 1-2 "Extract local observation data", Eq.18-19): the local observations of
 * every point of a PERIODIC Ny x Nx grid are gathered inside the library from the forecast
 * observations of the whole grid, so that Y_loc[M, Nx, l_max V] (5.3 times the state)
 * is never materialised.  For grid point (y, x) the local observations are the V observed
 * variables at the (2 hw + 1)^2 points of the square patch around it,
 *   local row j = v (2hw+1)^2 + (dy+hw)(2hw+1) + (dx+hw),  observed point (y+dy mod Ny, x+dx mod Nx),
 *   dY_j = Yf[v][yy][xx][:] - mean_m Yf[v][yy][xx][m]            Eq.18-19
 *   d_j  = yo[v][yy][xx] - mean_m Yf[v][yy][xx][m]
 *   r_j  = G(sqrt(dx^2+dy^2)) / sigma_o^2,  0 where obs_mask[yy][xx] == 0 (no observation there)
 * followed by the local analysis exactly as letkf_analysis_batched (same rho, same outputs).
 * G is the localisation function of PAPER.md:144 in grid units:
 *   loc_kind 0: Gaussian exp(-dist^2 / (2 loc_scale^2))            (BASELINE.json configs)
 *   loc_kind 1: Gaspari-Cohn (ref.[21]), half-width loc_scale, zero from 2 loc_scale on; the
 *               paper's cutoff 2(p-1) dx corresponds to loc_scale = p-1
 *
 *   Yf        in  [V][Ny][Nx][M]  forecast observations y_m^f = H x_m^f at every grid point
 *   yo        in  [V][Ny][Nx]     observations
 *   obs_mask  in  [Ny][Nx] bytes or NULL (NULL = every point observed)
 *   Xb        in  [Ny*Nx][nstate][M]   background ensemble, grid point index y*Nx + x
 *   Xa        out [Ny*Nx][nstate][M]   may alias Xb
 *   wbar      out [Ny*Nx][M] or NULL;  info out [Ny*Nx] or NULL
 *   work      >= letkf_analysis_grid_workspace_bytes(M, V, Ny, Nx, hw, nstate), or NULL
 * For M <= 64 and nstate <= 15 the gather runs inside the tridiagonalisation kernel (the field is
 * read through L2, nothing is materialised); otherwise Y_loc is materialised pass by pass in the
 * workspace and the any-M kernels are used.
 */
int letkf_analysis_grid(const double* Yf, const double* yo, const unsigned char* obs_mask,
                        const double* Xb, int M, int V, int Ny, int Nx, int nstate, int hw,
                        int loc_kind, double loc_scale, double sigma_o, double rho,
                        double* Xa, double* wbar, int* info,
                        void* work, size_t work_bytes, void* stream);

size_t letkf_analysis_grid_workspace_bytes(int M, int V, int Ny, int Nx, int hw, int nstate);

/*
 * The same two operations on HOST buffers (the end-to-end form: this is what bench.py's "e2e"
 * times).  Every array pointer is a HOST pointer with the layouts above; page-locked (pinned)
 * memory lets the copies run asynchronously at full PCIe rate, pageable memory works but
 * serialises them.  The library copies the batch in sub-chunk by sub-chunk on a copy-in stream,
 * starts each sub-chunk's kernels as soon as its own inputs have arrived, and reads each
 * sub-chunk's outputs back on a copy-out stream as soon as its last kernel is done.  The device staging
 * arena (inputs, outputs and workspace of one pass) is allocated on first use and KEPT by the
 * calling host thread for its next call, grown when a larger one is needed; letkf_host_release()
 * frees it.  The call BLOCKS
 * until the outputs are in the host buffers.  Return values as for the device forms (argument
 * positions are those of this signature); alignment of host pointers is not required.
 * V may alias A, Xa may alias Xb.  info / W / wbar may be NULL.
 */
int letkf_syev_batched_host(const double* A, int M, int batch, double* w, double* V, int* info);

int letkf_analysis_batched_host(const double* Yb, const double* d, const double* rinv_loc,
                                const double* Xb, int M, int p, int nstate, int batch, double rho,
                                double* Xa, double* W, double* wbar, int* info);

/* letkf_analysis_grid on HOST buffers: only the observation fields and the ensemble cross PCIe
 * (Y_loc never exists anywhere).  Argument positions as in this signature. */
int letkf_analysis_grid_host(const double* Yf, const double* yo, const unsigned char* obs_mask,
                             const double* Xb, int M, int V, int Ny, int Nx, int nstate, int hw,
                             int loc_kind, double loc_scale, double sigma_o, double rho,
                             double* Xa, double* wbar, int* info);

/* Frees the staging arena the host entry points keep for the calling host thread (no-op if none). */
void letkf_host_release(void);

/*
 * Measurement helper (not part of the method): runs `iters` dependent-chain-free fp64 FMA
 * rounds on every SM and writes one double per thread to `sink` (device, >= blocks*threads
 * doubles) so the work cannot be elided.  Returns the number of fp64 FMAs executed in
 * *fma_count (host pointer, may be NULL).  bench.py times it with CUDA events to obtain the
 * measured DFMA peak that the roofline fraction is quoted against.
 */
int letkf_probe_dfma(double* sink, int blocks, int threads, int iters,
                     unsigned long long* fma_count, void* stream);

/*
 * Profiling aid for bench.py (off by default; adds one CUDA event pair per kernel launch).
 * With profiling on, each compute call records events around every kernel it enqueues, on the
 * stream the kernel runs on, and counts the plane rotations its QL step generated.
 *   letkf_profile_enable(on)         switch; returns the previous setting.  on = 1: the call runs
 *                                    as ONE chunk on the caller's stream, so each record is a kernel
 *                                    timed alone; on = 2: the sub-chunk pipeline is kept and each
 *                                    record is taken on the private stream the kernel runs on (a
 *                                    timeline: records of different streams overlap)
 *   letkf_profile_record_start(i, &ms)   SYNCHRONISES; start of record i relative to record 0
 *   letkf_profile_count()            records held from the last compute call of this thread
 *   letkf_profile_record(i, &name, &ms)  SYNCHRONISES on record i's events; name is a static string
 *   letkf_profile_rotations()        SYNCHRONISES; total rotations generated by the last call
 */
int letkf_profile_enable(int on);
int letkf_profile_count(void);
int letkf_profile_record(int idx, const char** name, float* ms);
int letkf_profile_record_start(int idx, float* ms_from_first);
long long letkf_profile_rotations(void);
/* SYNCHRONISES; number of matrices of the last profiled call whose eigenvectors came from twisted
 * factorisations (no rotation logged or replayed) */
long long letkf_profile_direct(void);

/* Number of kernels the last compute call on this host thread enqueued (bench.py's
 * gpu_launches claim is counted from this, not guessed). */
int letkf_last_launch_count(void);

/* Test / experiment options (process-wide; every entry point takes ONE snapshot of them when it starts, so a
 * change from another host thread never takes effect in the middle of a call).  value -1 / 0 restores the default
 * where a default is "by size".
 *   "force_generic" 1: every M through the any-M kernels (otherwise only M > 160)
 *   "pipeline"      0: chunk after chunk on the caller's stream instead of the sub-chunk pipeline (default 1)
 *   "sub_chunk"     matrices per sub-chunk of the pipeline (0 = batch / 16, at least 512)
 *   "slots"         sub-chunks in flight = workspace slots (0 = all 16); "log_slots": of which as many may hold a
 *                   slot of the rotation log (0 = a 256 MB budget on the M <= 64 path, every slot elsewhere)
 *   "ql_tpb"        lanes per QL CTA: 32 / 64 / 96 / 128 / 192 (0 = 128 for M <= 64, 32 above)
 *   "two_pass"      QL log from a second, perfectly shifted pass: 0 / 1 (-1 = when batch x M >= 2^18)
 *   "log_shrink"    k divides the rotation-log capacity so that tests can force the in-kernel slow path
 *   "qform"         M <= 64: 1 = explicit Q formed by the reduction kernel, rotations replayed on its rows (round 1's
 *                   form); 0 (default) = reflectors kept, back-transform in the apply kernel
 *   "evec"          1 (default) = eigenvectors of T by twisted factorisations where the classifier allows (M <= 64 with
 *                   qform 0; M > 64 with bigvec 1); 0 = always the logged rotations
 *   "bigvec"        M > 64, evec 1: 1 (default) = the eigenvector route above 64 (eigenvectors of T in the matrix's record
 *                   of the rotation log, V = Q Z on the FP64 tensor cores); 0 = always the logged rotations
 *   "pack"          M <= 16, qform 0, EVD calls: two matrices per warp in the reduction and the apply kernel (1, default),
 *                   in the reduction only (2), in the apply kernel only (3), one matrix per warp (0)
 *   "bisect"        M <= 64, evec 1: eigenvalues by multisection with M threads per matrix: 0 / 1 (-1 = batch <= 1024)
 *   "pair"          32 < M <= 64: the reduction kernel takes two matrices per CTA: 0 / 1 (-1 = for 32 < M <= 48)
 *   "split"         48 < M <= 64: the reduction as two kernels, pivots M-1 ... 33 by two warps and the trailing
 *                   32 x 32 problem by one warp per matrix (default 1; 0 = one kernel)
 *   "mid_split"     64 < M <= 128: the reduction stops after pivot 64 and its trailing 64 x 64 block goes through the
 *                   register kernels of the M <= 64 path (1, default; 0 = one kernel down to pivot 1)
 *   "mid_reg"       64 < M <= 160: reduction with the matrix in shared memory (0) / in registers up to M = 128 and by the
 *                   any-M kernels above (1, default) / in registers (2)
 *   "host_pass"     matrices per pass of the host entry points (0 = what a 16 GiB staging arena holds)
 * Returns 0, or -1 for an unknown name. */
int letkf_set_option(const char* name, int value);

const char* letkf_status_string(int status);
int letkf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LETKF_H */

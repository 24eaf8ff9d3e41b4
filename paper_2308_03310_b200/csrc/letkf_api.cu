// letkf_api.cu -- the C ABI of libletkf (include/letkf.h): argument checking, workspace carving,
// dispatch on M, kernel launches.  No torch types; plain device pointers and sizes.
#include "../../include/letkf.h"

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <mutex>
#include <vector>

#include "common.cuh"
#include "ql_kernel.cuh"
#include "generic_kernels.cuh"
#include "fast_kernels.cuh"
#include "bisect_kernel.cuh"
#include "ns_kernel.cuh"
#include "mid_kernels.cuh"
#include "pack_kernels.cuh"
#include "big_kernels.cuh"
#include "gram_kernels.cuh"

namespace letkf {

static thread_local int g_launches = 0;

// ---- profiling aid (letkf_profile_*) --------------------------------------------------------
struct ProfRec { const char* name; cudaEvent_t e0, e1; };
struct Prof {
    bool on = false;
    bool keep_pipeline = false;   // letkf_profile_enable(2): time the kernels where they run
    std::vector<ProfRec> recs;
    std::vector<cudaEvent_t> pool;
    size_t used = 0;
    unsigned long long* d_rot = nullptr;
    cudaEvent_t get()
    {
        if (used == pool.size()) { cudaEvent_t e; cudaEventCreate(&e); pool.push_back(e); }
        return pool[used++];
    }
};
static thread_local Prof g_prof;

static void prof_reset(cudaStream_t st)
{
    g_prof.recs.clear();
    g_prof.used = 0;
    if (g_prof.on) {
        if (!g_prof.d_rot) cudaMalloc(&g_prof.d_rot, 2 * sizeof(unsigned long long));   // [0] rotations, [1] direct matrices
        cudaMemsetAsync(g_prof.d_rot, 0, 2 * sizeof(unsigned long long), st);
    }
}
static void prof_begin(const char* name, cudaStream_t st)
{
    if (!g_prof.on) return;
    ProfRec r{name, g_prof.get(), g_prof.get()};
    cudaEventRecord(r.e0, st);
    g_prof.recs.push_back(r);
}
static void prof_end(cudaStream_t st)
{
    if (!g_prof.on) return;
    cudaEventRecord(g_prof.recs.back().e1, st);
}

#define KLAUNCH(name, st, ...)                                 \
    do {                                                       \
        prof_begin(name, st);                                  \
        __VA_ARGS__;                                           \
        prof_end(st);                                          \
        cudaError_t e_ = cudaGetLastError();                   \
        if (e_ != cudaSuccess) return (int)e_;                 \
        ++g_launches;                                          \
    } while (0)

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ---- options (letkf_set_option) ------------------------------------------------------------------
// Process-wide settings, written under a mutex.  Every entry point takes ONE snapshot into the
// calling thread's copy when it starts and reads nothing else, so a letkf_set_option from another
// host thread can never change the layout or the kernel choice in the middle of a call.
struct Options {
    int force_generic = 0;   // 1: every M through the any-M kernels (tests)
    int pipeline = 1;        // 0: one chunk at a time on the caller's stream
    int sub_chunk = 0;       // matrices per sub-chunk of the pipeline (0 = by size)
    int slots = 0;           // sub-chunks in flight = workspace slots (0 = default)
    int log_slots = 0;       // of which as many may be between the start of their QL and the end of their apply
                             // kernel (slots of the rotation log, the large part of a slot; 0 = default)
    int mid_reg = 1;         // 64 < M <= 160 reduced in shared memory (0) / registers up to M = 128 (1) / registers (2)
    int log_shrink = 1;      // divides the rotation-log capacity (tests force the slow path)
    int ql_tpb = 0;          // matrices per QL CTA (0 = by size)
    int two_pass = -1;       // QL with a second, perfectly shifted pass: -1 = by batch size, 0 / 1
    int host_pass = 0;       // matrices per pass of the host entry points (0 = by arena size; tests)
    int qform = 0;           // M <= 64: 1 = explicit Q formed by the reduction kernel and replayed on (through the
                             // output buffer); 0 = reflectors kept, eigenvectors of T formed in the apply kernel,
                             // which then does the back-transform (nothing but the reflectors crosses HBM in between)
    int bisect = -1;         // M <= 64, evec = 1: eigenvalues by multisection with M threads per matrix instead of the QL
                             // kernel's one (the latency regime): -1 = for batches up to BISECT_MAX_BATCH, 0 / 1
    int pair = -1;           // 32 < M <= 64, qform = 0: a CTA reduces two matrices, their trailing 32 x 32 blocks side by
                             // side on its two warps (0: one matrix per CTA, the second warp idle through the last 32
                             // pivots).  -1 = where it measured faster: 32 < M <= 48 without the Gram step (config 5,
                             // M = 48: 1.74 -> 1.51 ms; at M = 64 the paired kernel spills and loses, 1.46 -> 1.65 ms)
    int split = 1;           // 48 < M <= 64, qform = 0: the reduction as two kernels (pivots down to 33 by two warps,
                             // the trailing 32 x 32 problem by one warp per matrix): 1.07 + 0.25 ms against 1.46 ms (config 3)
    int pack = 1;            // M <= 16, qform = 0, EVD calls: two matrices per warp (pack_kernels.cuh): 1 = reduction and
                             // apply kernel, 2 = reduction only, 3 = apply kernel only, 0 = one matrix per warp
    int mid_split = 1;       // 64 < M <= 128, mid_reg >= 1: the reduction stops after pivot 64 and the trailing 64 x 64 block goes
                             // through the register kernels of the M <= 64 path (0 = one kernel down to pivot 1)
    int bigvec = 1;          // M > 64 (and evec = 1): eigenvectors of T by twisted factorisations and V = Q Z as one product on
                             // the FP64 tensor cores where the spectrum allows (big_kernels.cuh); 0 = always the rotation log
    int evec = 1;            // M <= 64, qform = 0: 1 = eigenvectors of T by twisted factorisations where the spectrum
                             // allows (ql_log_kernel classifies), the logged rotations otherwise; 0 = always the log
};
static Options g_options;
static std::mutex g_options_mu;
static thread_local Options t_opt;
static thread_local int t_depth = 0;
struct EntryScope {                      // first thing every entry point constructs
    EntryScope()
    {
        if (t_depth++ == 0) { std::lock_guard<std::mutex> lk(g_options_mu); t_opt = g_options; }
    }
    ~EntryScope() { --t_depth; }
};

// ---- workspace -------------------------------------------------------------------------------------
// The workspace holds `nslot` slots of `per` matrices each; sub-chunk k of a call lives in slot
// k mod nslot for as long as its three kernels are in flight (Streams).  The
// rotation log (with its sweep headers: 72 of the 93 KB a matrix of order 64 needs) is only touched
// from the QL kernel on, so it has slots of its own, `nlog` <= nslot of them: the reductions may run
// ahead of the eigensolver without holding log space.
static bool use_fast(int M) { return fast_supported(M) && !t_opt.force_generic; }
static bool use_mid(int M) { return mid_supported(M) && !t_opt.force_generic; }
// M > 64: the eigenvector route of big_kernels.cuh (Z in the matrix's record of the rotation log, which must have its full size)
static bool use_bigvec(int M) { return M > 64 && !use_fast(M) && t_opt.evec && t_opt.bigvec && t_opt.log_shrink == 1; }
// 64 < M <= 128: the reduction hands its trailing 64 x 64 block to the register kernels (mid_kernels.cuh, HEAD)
static bool use_midsplit(int M)
{
    return use_mid(M) && mid_threads(M) <= 128 && t_opt.mid_reg >= 1 && t_opt.mid_split && t_opt.log_shrink == 1;
}
static bool use_getvec(int M) { return (use_fast(M) && !t_opt.qform && t_opt.evec) || use_bigvec(M); }

static size_t carve(Workspace& ws, void* base, int M, int nmat, int nlogmat, bool two_pass)
{
    char* p = reinterpret_cast<char*>(base);
    size_t off = 0;
    auto take = [&](size_t bytes) { char* q = p ? p + off : nullptr; off = align_up(off + bytes, 256); return q; };
    ws.swcap = sweep_capacity(M);
    ws.logcap = log_capacity(M, two_pass) / t_opt.log_shrink;      // (the memory is still sized for the full log)
    ws.reflstride = (use_fast(M) && !t_opt.qform) ? fast_refl_doubles(M) : (use_midsplit(M) ? ((mid_split_refl_doubles(M) + 1) & ~1) : 0);
    ws.rot_counter = g_prof.on ? g_prof.d_rot : nullptr;
    ws.dws     = reinterpret_cast<double*>(take(sizeof(double) * (size_t)M * nmat));
    ws.ews     = reinterpret_cast<double*>(take(sizeof(double) * (size_t)M * nmat));
    ws.perm    = reinterpret_cast<int*>(take(sizeof(int) * (size_t)M * nmat));
    ws.nsweeps = reinterpret_cast<int*>(take(sizeof(int) * (size_t)nmat));
    ws.flags   = reinterpret_cast<int*>(take(sizeof(int) * (size_t)nmat));
    ws.hdr     = reinterpret_cast<uint32_t*>(take(sizeof(uint32_t) * (size_t)ws.swcap * nlogmat));
    ws.rot     = reinterpret_cast<double2*>(take(sizeof(double2) * (size_t)log_capacity(M, two_pass) * nlogmat));
    ws.refl    = reinterpret_cast<double*>(take(sizeof(double) * (size_t)ws.reflstride * nmat));
    ws.s1      = reinterpret_cast<double*>(take(use_getvec(M) ? sizeof(double) * (size_t)M * nmat : 0));
    return off;
}

// the records of a sub-chunk: matrices b0 ... of the small arrays, l0 ... of the log arrays
static Workspace ws_slice(const Workspace& w, int M, int b0, int l0)
{
    Workspace s = w;
    s.dws += (size_t)b0 * M;
    s.ews += (size_t)b0 * M;
    s.perm += (size_t)b0 * M;
    s.nsweeps += b0;
    s.flags += b0;
    s.hdr += (size_t)l0 * w.swcap;
    s.rot += (size_t)l0 * w.logcap;
    s.refl += (size_t)b0 * w.reflstride;
    if (s.s1) s.s1 += (size_t)b0 * M;
    return s;
}

// How a call over `batch` matrices is cut up.  Pipelined: nsub sub-chunks of `per` matrices flow
// tridiag -> QL -> apply over private streams, at most `nslot` of them in flight (a slot of the
// workspace each).  Not pipelined (small batches, pipeline = 0, kernel-alone profiling): chunks of
// `per` matrices one after the other on the caller's stream.
struct Plan { int per, nslot, nlog, nsub; bool pipelined, two_pass; int ql_mode; bool bisect; };
static const int BISECT_MAX_BATCH = 1024;
static const int PIPE_MIN_SUB = 512;     // smallest sub-chunk worth launches of its own
static const int PIPE_MAX_SUBS = 16;     // sub-chunks per call (bounds the launch count)
static const int PIPE_SLOTS = 16;        // default number of sub-chunks in flight: all of them
static const size_t PIPE_LOG_BYTES = (size_t)256 << 20;   // default size of the log slots together
static const int NQ_STREAMS = 16;
#ifndef LETKF_NT_STREAMS
#define LETKF_NT_STREAMS 4
#endif
#ifndef LETKF_NA_STREAMS
#define LETKF_NA_STREAMS 4
#endif
static const int NT_STREAMS = LETKF_NT_STREAMS, NA_STREAMS = LETKF_NA_STREAMS;

static int round_up(int x, int a) { return (x + a - 1) / a * a; }

// bytes of a workspace for nmat matrices in flight (the one formula every size query and every check uses)
static size_t plan_bytes(int M, size_t nmat, size_t nlogmat, size_t extra, bool two_pass)
{
    Workspace tmp;
    return carve(tmp, nullptr, M, (int)nmat, (int)nlogmat, two_pass) + nmat * extra + 6 * 256;
}

// extra: bytes per matrix the caller keeps per slot beside the EVD workspace (analysis: Q/V, lam, g, gathered Y_loc);
// avail: bytes of the workspace at hand (0: plan for the recommended size)
static Plan make_plan(int M, int batch, size_t extra, size_t avail)
{
    Plan pl;
    pl.two_pass = t_opt.two_pass >= 0 ? t_opt.two_pass != 0 : ((long)batch * M >= (1L << 18));
    pl.ql_mode = pl.two_pass ? QL_TWO_PASS : QL_ONE_PASS;
    // (a logged pass is always the second one.  M > 128: scout and logger side by side and the classification at the end --
    // measured, config 5 with p = 98, where every matrix of M >= 128 stays on the log: M = 256 27.7 ms against 28.9 ms for
    // classify-then-log; at M = 96, where none does, 8.5 against 8.0 ms)
    if (use_getvec(M)) { pl.ql_mode = (use_bigvec(M) && M > 128) ? QL_PAIRED_CLASSIFY : QL_CLASSIFY; pl.two_pass = true; }
    pl.bisect = use_getvec(M) && use_fast(M) && (t_opt.bisect >= 0 ? t_opt.bisect != 0 : batch <= BISECT_MAX_BATCH);
    // (M > 160: the kernels of the any-M path hold two CTAs per SM -- sub-chunks of one full wave, measured M = 256: 18.8 -> 17.9 ms)
    const int min_sub = M > 160 ? 296 : PIPE_MIN_SUB;
    const bool want_pipe = t_opt.pipeline && (!g_prof.on || g_prof.keep_pipeline) && batch >= 2 * min_sub;
    auto bytes_for = [&](size_t n, size_t nl) { return plan_bytes(M, n, nl, extra, pl.two_pass); };
    if (want_pipe) {
        int per = t_opt.sub_chunk > 0 ? t_opt.sub_chunk : round_up((batch + PIPE_MAX_SUBS - 1) / PIPE_MAX_SUBS, 64);
        if (per < min_sub && t_opt.sub_chunk <= 0) per = min_sub;
        if (per > batch) per = batch;
        int nsub = (batch + per - 1) / per;
        int nslot = t_opt.slots > 0 ? t_opt.slots : PIPE_SLOTS;
        if (nslot > nsub) nslot = nsub;
        const size_t log_entry = sizeof(double2) * (size_t)log_capacity(M, pl.two_pass) + sizeof(uint32_t) * (size_t)sweep_capacity(M);
        // where every matrix logs its rotations (M > 64, or evec = 0) each slot has its log; where most
        // matrices never do (the eigenvector path of M <= 64) the log slots share a fixed budget
        int nlog = t_opt.log_slots > 0 ? t_opt.log_slots
                 : ((pl.ql_mode == QL_CLASSIFY && use_fast(M)) ? (int)((PIPE_LOG_BYTES + log_entry * per - 1) / (log_entry * per)) : nslot);
        if (nlog < 2) nlog = 2;
        if (nlog > nslot) nlog = nslot;
        if (avail) {                       // a smaller workspace: fewer log slots first, then fewer slots
            while (nlog > 2 && bytes_for((size_t)per * nslot, (size_t)per * nlog) > avail) --nlog;
            while (nslot > 2 && bytes_for((size_t)per * nslot, (size_t)per * nlog) > avail) { --nslot; if (nlog > nslot) nlog = nslot; }
        }
        if (nslot >= 2 && (!avail || bytes_for((size_t)per * nslot, (size_t)per * nlog) <= avail)) {
            pl.per = per; pl.nslot = nslot; pl.nlog = nlog; pl.nsub = nsub; pl.pipelined = true;
            return pl;
        }
    }
    // sequential chunks: as large as the workspace allows (recommended: what the pipeline would take)
    int per = batch;
    if (avail) {
        while (per > 1 && bytes_for((size_t)per, (size_t)per) > avail) per = (per + 1) / 2;
    } else {
        const int cap = round_up((batch + PIPE_MAX_SUBS - 1) / PIPE_MAX_SUBS, 64) * 4;
        if (per > cap && cap >= 2 * PIPE_MIN_SUB) per = cap;
    }
    pl.per = per; pl.nslot = 1; pl.nlog = 1; pl.nsub = (batch + per - 1) / per; pl.pipelined = false;
    return pl;
}

static inline bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

template <typename K>
static cudaError_t allow_smem(K kernel, size_t bytes)
{
    cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (bytes <= 48 * 1024) return cudaSuccess;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// a1/a2 inputs when the matrix is to be formed from the LETKF observations instead of read
struct GramArgs { const double* Yb; const double* d; const double* r; int p; double shift; double* gout; GridArgs grid; };

template <int MT, bool QFORM>
static int fast_tridiag_run(const double* A, double* V, Workspace ws, int M, int n, cudaStream_t st, const GramArgs* gram)
{
    const size_t smem = fast_tridiag_smem<MT>();
    cudaError_t ce;
    if constexpr (MT == 64 && !QFORM) {
        if (t_opt.split && M > 48) {
            if (gram) {
                if ((ce = allow_smem(fast_tridiag<MT, true, false, double, true>, smem)) != cudaSuccess) return (int)ce;
                KLAUNCH("fast_tridiag_head<gram>", st,
                        (fast_tridiag<MT, true, false, double, true><<<n, FastCfg<MT>::NT, smem, st>>>(
                            static_cast<const double*>(nullptr), V, ws, M, gram->Yb, gram->d, gram->r, gram->p, gram->shift, gram->gout, gram->grid, n)));
            } else {
                if ((ce = allow_smem(fast_tridiag<MT, false, false, double, true>, smem)) != cudaSuccess) return (int)ce;
                KLAUNCH("fast_tridiag_head", st,
                        (fast_tridiag<MT, false, false, double, true><<<n, FastCfg<MT>::NT, smem, st>>>(
                            A, V, ws, M, nullptr, nullptr, nullptr, 0, 0.0, nullptr, GridArgs{}, n)));
            }
            KLAUNCH("fast_tridiag_tail", st, fast_tridiag_tail<double><<<n, 32, fast_tridiag_tail_smem<double>(), st>>>(ws, M));
            return 0;
        }
    }
    if constexpr ((MT == 64 || MT == 48) && !QFORM) {
        if (t_opt.pair > 0 || (t_opt.pair < 0 && MT == 48 && !gram)) {
            const size_t ps = fast_tridiag_smem_pair<MT, double, true>();
            if (gram) {
                if ((ce = allow_smem(fast_tridiag<MT, true, false, double, false, true>, ps)) != cudaSuccess) return (int)ce;
                KLAUNCH("fast_tridiag<gram>", st,
                        (fast_tridiag<MT, true, false, double, false, true><<<(n + 1) / 2, FastCfg<MT>::NT, ps, st>>>(
                            static_cast<const double*>(nullptr), V, ws, M, gram->Yb, gram->d, gram->r, gram->p, gram->shift, gram->gout, gram->grid, n)));
            } else {
                if ((ce = allow_smem(fast_tridiag<MT, false, false, double, false, true>, ps)) != cudaSuccess) return (int)ce;
                KLAUNCH("fast_tridiag", st,
                        (fast_tridiag<MT, false, false, double, false, true><<<(n + 1) / 2, FastCfg<MT>::NT, ps, st>>>(
                            A, V, ws, M, nullptr, nullptr, nullptr, 0, 0.0, nullptr, GridArgs{}, n)));
            }
            return 0;
        }
    }
    if (gram) {
        if ((ce = allow_smem(fast_tridiag<MT, true, QFORM>, smem)) != cudaSuccess) return (int)ce;
        KLAUNCH("fast_tridiag<gram>", st,
                fast_tridiag<MT, true, QFORM><<<n, FastCfg<MT>::NT, smem, st>>>(
                    static_cast<const double*>(nullptr), V, ws, M, gram->Yb, gram->d, gram->r, gram->p, gram->shift, gram->gout, gram->grid, n));
    } else {
        if ((ce = allow_smem(fast_tridiag<MT, false, QFORM>, smem)) != cudaSuccess) return (int)ce;
        KLAUNCH("fast_tridiag", st,
                fast_tridiag<MT, false, QFORM><<<n, FastCfg<MT>::NT, smem, st>>>(
                    A, V, ws, M, nullptr, nullptr, nullptr, 0, 0.0, nullptr, GridArgs{}, n));
    }
    return 0;
}

template <int MT, bool QFORM>
static int fast_apply_run(double* V, double* w, int* info, Workspace ws, int M, int n, cudaStream_t st, const EpiArgs* ep)
{
    cudaError_t ce;
    if (ep) {
        const size_t smem = fast_apply_smem<MT>(ws.swcap, ep->ns, QFORM);
        if ((ce = allow_smem(fast_apply<MT, true, QFORM>, smem)) != cudaSuccess) return (int)ce;
        KLAUNCH("fast_apply<epilogue>", st, fast_apply<MT, true, QFORM><<<n, FastCfg<MT>::NT, smem, st>>>(V, w, info, ws, M, *ep));
    } else {
        const size_t smem = fast_apply_smem<MT>(ws.swcap, 0, QFORM);
        if ((ce = allow_smem(fast_apply<MT, false, QFORM>, smem)) != cudaSuccess) return (int)ce;
        KLAUNCH("fast_apply", st, fast_apply<MT, false, QFORM><<<n, FastCfg<MT>::NT, smem, st>>>(V, w, info, ws, M, EpiArgs{}));
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// The EVD of n matrices as three stages.  stage_T: a3 (+ a1, a2 with `gram`) -- M <= 64: (d, e) and
// the reflectors into the workspace; above: (d, e) and the explicit Q^T into V.  stage_QL: a4, the
// logged QL iteration.  stage_AP: a5, replay of the log (and back-transform), eigenvalue sort.
// ws is the workspace slice of these n matrices.
static int stage_T(const double* A, int M, int n, double* V, Workspace ws, cudaStream_t st,
                   const GramArgs* gram)
{
    if (use_fast(M) && M <= 16 && !gram && !t_opt.qform && (t_opt.pack == 1 || t_opt.pack == 2)) {
        KLAUNCH("pack16_tridiag", st,
                (pack16_tridiag<<<(n + 2 * PK_WARPS - 1) / (2 * PK_WARPS), 32 * PK_WARPS, pack16_tridiag_smem(), st>>>(A, ws, M, n)));
        return 0;
    }
    if (use_fast(M)) {
        if (t_opt.qform) {
            switch (fast_bucket(M)) {
                case 16: return fast_tridiag_run<16, true>(A, V, ws, M, n, st, gram);
                case 32: return fast_tridiag_run<32, true>(A, V, ws, M, n, st, gram);
                case 48: return fast_tridiag_run<48, true>(A, V, ws, M, n, st, gram);
                default: return fast_tridiag_run<64, true>(A, V, ws, M, n, st, gram);
            }
        }
        switch (fast_bucket(M)) {
            case 16: return fast_tridiag_run<16, false>(A, V, ws, M, n, st, gram);
            case 32: return fast_tridiag_run<32, false>(A, V, ws, M, n, st, gram);
            case 48: return fast_tridiag_run<48, false>(A, V, ws, M, n, st, gram);
            default: return fast_tridiag_run<64, false>(A, V, ws, M, n, st, gram);
        }
    }
    if (gram) {
        if (M > 64) {                                         // the contraction on the FP64 tensor cores (gram_kernels.cuh)
            cudaError_t ge;
            const size_t gs = gram_smem(M, gram->p);
            if ((ge = allow_smem(big_gram, gs)) != cudaSuccess) return (int)ge;
            KLAUNCH("big_gram", st,
                    big_gram<<<n, GRAM_NT, gs, st>>>(gram->Yb, gram->d, gram->r, M, gram->p, gram_chunk(M, gram->p), gram->shift, V, gram->gout));
        } else
        KLAUNCH("generic_gram", st,
                generic_gram<<<n, 256, 0, st>>>(gram->Yb, gram->d, gram->r, M, gram->p, gram->shift, V, gram->gout));
        A = V;
    }
    // (128 < M <= 160: the any-M reduction below, 7.1 + 3.0 ms at M = 160 against 10.5 ms for the shared-memory one; the
    // replay stays mid_apply's)
    if (use_mid(M) && (M <= 128 || t_opt.mid_reg == 0 || t_opt.mid_reg == 2)) {   // matrix resident in registers / shared memory
        cudaError_t ce;
        const size_t smem = mid_tridiag_smem(M);
        const int mt = mid_threads(M);
        // registers hold the matrix up to M = 128 (measured, batch 2^26/M^2: M = 96 6.58 -> 5.12 ms, M = 128 9.42 -> 7.57 ms);
        // at MT = 160 the 80 matrix registers of a thread spill under the 102 a CTA of 640 allows and
        // the shared-memory form is as fast (10.5 vs 10.9 ms): mid_reg = 1 (default) / 2 (force) / 0 (never)
        const bool reg = t_opt.mid_reg == 2 || (t_opt.mid_reg == 1 && mt <= 128);
        if (use_midsplit(M)) {
            // pivots M-1 ... 64 here, the trailing 64 x 64 block in the register kernels, then Q^T from both sets of
            // reflectors.  Scratch (free until the QL kernel): the block, its d and e, flat in the rotation-log area
            double* blk = reinterpret_cast<double*>(ws.rot);
            double* d64 = blk + (size_t)n * 4096;
            double* e64 = d64 + (size_t)n * 64;
            auto head = mt == 96 ? mid_tridiag_formq_reg<96, true> : mid_tridiag_formq_reg<128, true>;
            if ((ce = allow_smem(head, smem)) != cudaSuccess) return (int)ce;
            KLAUNCH("mid_tridiag_head", st, head<<<n, MID_TPR * mt, smem, st>>>(A, V, ws, M));
            Workspace wsv = ws;
            wsv.dws = d64; wsv.ews = e64;
            int rc = fast_tridiag_run<64, false>(blk, nullptr, wsv, 64, n, st, nullptr);
            if (rc) return rc;
            auto fq = mt == 96 ? mid_formq_split<96> : mid_formq_split<128>;
            if ((ce = allow_smem(fq, smem)) != cudaSuccess) return (int)ce;
            KLAUNCH("mid_formq_split", st, fq<<<n, MID_TPR * mt, smem, st>>>(V, ws, M, d64, e64));
            return 0;
        }
        auto kern = reg ? (mt == 96 ? mid_tridiag_formq_reg<96> : (mt == 128 ? mid_tridiag_formq_reg<128> : mid_tridiag_formq_reg<160>))
                        : (mt == 96 ? mid_tridiag_formq<96> : (mt == 128 ? mid_tridiag_formq<128> : mid_tridiag_formq<160>));
        if ((ce = allow_smem(kern, smem)) != cudaSuccess) return (int)ce;
        KLAUNCH("mid_tridiag_formq", st, kern<<<n, MID_TPR * mt, smem, st>>>(A, V, ws, M));
        return 0;
    }
    const size_t td_smem = sizeof(double) * ((4 + GEN_QK + 1) * (size_t)M + GEN_NT / 32);   // v, w, p, taus; vk[GEN_QK][M] shared with v' + pT[8][M]
    // two launches of one kernel (phase 1: the reduction, phase 2: Q^T from the reflectors), so that each shows in the records
    KLAUNCH("generic_tridiag", st, generic_tridiag_formq<1><<<n, GEN_NT, td_smem, st>>>(A, V, ws, M));
    if (M <= 192) KLAUNCH("generic_formq", st, (generic_tridiag_formq<2, 6><<<n, GEN_NT, td_smem, st>>>(A, V, ws, M)));
    else if (M <= 224) KLAUNCH("generic_formq", st, (generic_tridiag_formq<2, 7><<<n, GEN_NT, td_smem, st>>>(A, V, ws, M)));
    else KLAUNCH("generic_formq", st, (generic_tridiag_formq<2, 8><<<n, GEN_NT, td_smem, st>>>(A, V, ws, M)));
    return 0;
}

template <int TPB, int MODE>
static int ql_launch(int M, int n, double* w, int* info, Workspace ws, cudaStream_t st)
{
    cudaError_t ce;
    const size_t ql_smem = sizeof(double) * 2 * (size_t)M * TPB + (8 * (size_t)((M + 63) / 64) + 16) * TPB;   // (d, e) per lane + block boundaries, threshold, sort state
    if ((ce = allow_smem(ql_log_kernel<TPB, MODE>, ql_smem)) != cudaSuccess) return (int)ce;
    const int per_cta = (MODE == QL_TWO_PASS || MODE == QL_LOGPASS_PAIRED || MODE == QL_PAIRED_CLASSIFY) ? TPB / 2 : TPB;  // two lanes per matrix when the iteration runs twice side by side
    const int qblocks = (n + per_cta - 1) / per_cta;
    KLAUNCH("ql_log_kernel", st, (ql_log_kernel<TPB, MODE><<<qblocks, TPB, ql_smem, st>>>(ws, M, n, w, info)));
    return 0;
}
template <int TPB>
static int ql_run(int M, int n, double* w, int* info, Workspace ws, cudaStream_t st, int mode)
{
    switch (mode) {
        case QL_TWO_PASS: return ql_launch<TPB, QL_TWO_PASS>(M, n, w, info, ws, st);
        case QL_CLASSIFY: return ql_launch<TPB, QL_CLASSIFY>(M, n, w, info, ws, st);
        case QL_PAIRED_CLASSIFY: return ql_launch<TPB, QL_PAIRED_CLASSIFY>(M, n, w, info, ws, st);
        case QL_LOGPASS: return ql_launch<TPB, QL_LOGPASS>(M, n, w, info, ws, st);
        case QL_LOGPASS_PAIRED: return ql_launch<TPB, QL_LOGPASS_PAIRED>(M, n, w, info, ws, st);
        default: return ql_launch<TPB, QL_ONE_PASS>(M, n, w, info, ws, st);
    }
}

static int stage_QL(int M, int n, double* w, int* info, Workspace ws, cudaStream_t st, int mode)
{
    int tpb = t_opt.ql_tpb ? t_opt.ql_tpb : (M <= 64 ? 128 : 32);
    while (tpb > 32 && (sizeof(double) * 2 * (size_t)M + 48) * tpb > 200 * 1024) tpb -= 32;
    switch (tpb) {
        case 192: return ql_run<192>(M, n, w, info, ws, st, mode);
        case 128: return ql_run<128>(M, n, w, info, ws, st, mode);
        case 96: return ql_run<96>(M, n, w, info, ws, st, mode);
        case 64: return ql_run<64>(M, n, w, info, ws, st, mode);
        default: return ql_run<32>(M, n, w, info, ws, st, mode);
    }
}

// a4 for small batches (bisect_kernel.cuh): eigenvalues by multisection, M threads per matrix, then the
// same classification as QL_CLASSIFY
static int stage_bisect(int M, int n, double* w, int* info, Workspace ws, cudaStream_t st)
{
    switch (fast_bucket(M)) {
        case 16: KLAUNCH("bisect_classify_kernel", st, bisect_classify_kernel<16><<<n, FastCfg<16>::NT, 0, st>>>(ws, M, w, info)); break;
        case 32: KLAUNCH("bisect_classify_kernel", st, bisect_classify_kernel<32><<<n, FastCfg<32>::NT, 0, st>>>(ws, M, w, info)); break;
        case 48: KLAUNCH("bisect_classify_kernel", st, bisect_classify_kernel<48><<<n, FastCfg<48>::NT, 0, st>>>(ws, M, w, info)); break;
        default: KLAUNCH("bisect_classify_kernel", st, bisect_classify_kernel<64><<<n, FastCfg<64>::NT, 0, st>>>(ws, M, w, info)); break;
    }
    return 0;
}

// the logging pass of the matrices QL_CLASSIFY left pending (the first kernel to touch the log slot)
static int stage_QLlog(int M, int n, double* w, int* info, Workspace ws, cudaStream_t st, bool paired)
{
    return stage_QL(M, n, w, info, ws, st, paired ? QL_LOGPASS_PAIRED : QL_LOGPASS);
}

static int stage_AP(int M, int n, double* w, double* V, int* info, Workspace ws, cudaStream_t st,
                    const EpiArgs* ep = nullptr)
{
    const size_t ap_smem = sizeof(double) * (5 * (size_t)M + 2 * 32 * 33);
    if (use_fast(M) && M <= 16 && !ep && !t_opt.qform && (t_opt.pack == 1 || t_opt.pack == 3)) {
        KLAUNCH("pack16_apply", st,
                (pack16_apply<<<(n + 2 * PK_WARPS - 1) / (2 * PK_WARPS), 32 * PK_WARPS, pack16_apply_smem(), st>>>(V, w, info, ws, M, n)));
        return 0;
    }
    if (use_fast(M)) {      // (matrices whose rotation log is unusable are finished inside the kernel)
        if (t_opt.qform) {
            switch (fast_bucket(M)) {
                case 16: return fast_apply_run<16, true>(V, w, info, ws, M, n, st, ep);
                case 32: return fast_apply_run<32, true>(V, w, info, ws, M, n, st, ep);
                case 48: return fast_apply_run<48, true>(V, w, info, ws, M, n, st, ep);
                default: return fast_apply_run<64, true>(V, w, info, ws, M, n, st, ep);
            }
        }
        switch (fast_bucket(M)) {
            case 16: return fast_apply_run<16, false>(V, w, info, ws, M, n, st, ep);
            case 32: return fast_apply_run<32, false>(V, w, info, ws, M, n, st, ep);
            case 48: return fast_apply_run<48, false>(V, w, info, ws, M, n, st, ep);
            default: return fast_apply_run<64, false>(V, w, info, ws, M, n, st, ep);
        }
    }
    if (use_bigvec(M)) {    // the matrices the classifier left to the eigenvector route (the kernels below skip them)
        cudaError_t ce;
        if ((ce = allow_smem(big_getvec, big_getvec_smem(M))) != cudaSuccess) return (int)ce;
        KLAUNCH("big_getvec", st, big_getvec<<<n, (M + 31) / 32 * 32, big_getvec_smem(M), st>>>(ws, w, M));
#define LETKF_BIG_GEMM(RTW, CT)                                                                               \
        do {                                                                                                  \
            if ((ce = allow_smem(big_gemm<RTW, CT>, big_gemm_smem<CT>(M))) != cudaSuccess) return (int)ce;    \
            KLAUNCH("big_gemm", st, (big_gemm<RTW, CT><<<n, BIG_NT, big_gemm_smem<CT>(M), st>>>(V, ws, M))); \
        } while (0)
        if (M <= 96) LETKF_BIG_GEMM(2, 12);
        else if (M <= 128) LETKF_BIG_GEMM(2, 16);
        else if (M <= 160) LETKF_BIG_GEMM(3, 10);
        else if (M <= 192) LETKF_BIG_GEMM(3, 8);
        else LETKF_BIG_GEMM(4, 8);
#undef LETKF_BIG_GEMM
    }
    if (use_mid(M)) {
        cudaError_t ce;
        const int ms = mid_apply_round(M, ws.swcap);
        const size_t smem = mid_apply_smem(M, ws.swcap, ms);
        if ((ce = allow_smem(mid_apply, smem)) != cudaSuccess) return (int)ce;
        const int nsplit = mid_apply_split(M), ncol = mid_apply_cols(M);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)n * nsplit);
        cfg.blockDim = dim3((ncol + 31) / 32 * 32);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = nsplit; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        KLAUNCH("mid_apply", st, cudaLaunchKernelEx(&cfg, mid_apply, V, ws, M, ms, nsplit, ncol));
        // finisher for matrices whose rotation log overflowed (normally none: a few CTAs scan the flags and exit)
        KLAUNCH("generic_apply(flagged)", st,
                generic_apply<<<(n + GEN_NT - 1) / GEN_NT < 8 ? (n + GEN_NT - 1) / GEN_NT : 8, GEN_NT, ap_smem, st>>>(
                    V, w, ws, M, n, info, /*only_flagged=*/1, /*q_rowmajor=*/0));
        return 0;
    }
    const int ap_nt = M <= 32 ? 64 : (M + 31) / 32 * 32;          // thread r = column r of Q^T: no idle warps (M = 192: 5.6 -> 4.7 ms)
    KLAUNCH("generic_apply", st, generic_apply<<<n, ap_nt, ap_smem, st>>>(V, w, ws, M, n, info, 0, 0));
    return 0;
}

// ---------------------------------------------------------------------------------------------
// Private streams of the calling host thread.  A call over n matrices is cut into sub-chunks that
// flow through three stages on separate streams: ql_log_kernel is bound by the serial latency of
// one matrix's iteration and keeps one warp per SM sub-partition busy at most, so it runs beside
// the ALU-bound stage_T / stage_AP kernels of the neighbouring sub-chunks (highest priority, so a
// ready QL block takes the first free slot).  stage_T outranks stage_AP: every QL kernel should
// start as early as possible, the apply kernels fill the machine behind them.  Everything is forked
// from and joined back into the caller's stream with events: the caller sees plain stream order.
struct Pipe {
    int dev = -1;
    cudaStream_t sT[NT_STREAMS] = {}, sA[NA_STREAMS] = {};
    cudaStream_t sQ[NQ_STREAMS] = {};
    std::vector<cudaEvent_t> ev;
    size_t used = 0;
    void destroy()
    {
        for (auto& s : sT) if (s) { cudaStreamDestroy(s); s = nullptr; }
        for (auto& s : sA) if (s) { cudaStreamDestroy(s); s = nullptr; }
        for (auto& s : sQ) if (s) { cudaStreamDestroy(s); s = nullptr; }
        for (auto e : ev) cudaEventDestroy(e);
        ev.clear();
        used = 0;
        dev = -1;
    }
    int init()
    {
        int d = 0;
        cudaError_t ce = cudaGetDevice(&d);
        if (ce != cudaSuccess) return (int)ce;
        if (d == dev) return 0;
        if (dev >= 0) {                       // the thread moved to another device: drop the old streams
            cudaSetDevice(dev);
            destroy();
            cudaSetDevice(d);
        }
        int least = 0, greatest = 0;
        cudaDeviceGetStreamPriorityRange(&least, &greatest);
        const int mid = (greatest < least) ? greatest + 1 : greatest;
        for (int k = 0; k < NT_STREAMS; ++k)
            if ((ce = cudaStreamCreateWithPriority(&sT[k], cudaStreamNonBlocking, mid)) != cudaSuccess) return (int)ce;
        for (int k = 0; k < NA_STREAMS; ++k)
            if ((ce = cudaStreamCreateWithPriority(&sA[k], cudaStreamNonBlocking, least)) != cudaSuccess) return (int)ce;
        for (int k = 0; k < NQ_STREAMS; ++k)
            if ((ce = cudaStreamCreateWithPriority(&sQ[k], cudaStreamNonBlocking, greatest)) != cudaSuccess) return (int)ce;
        dev = d;
        return 0;
    }
    cudaEvent_t event()
    {
        if (used == ev.size()) {
            cudaEvent_t e = nullptr;
            cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
            ev.push_back(e);
        }
        return ev[used++];
    }
    // `to` waits for everything enqueued on `from` so far
    int link(cudaStream_t from, cudaStream_t to)
    {
        cudaEvent_t e = event();
        cudaError_t ce;
        if (!e) return (int)cudaErrorMemoryAllocation;
        if ((ce = cudaEventRecord(e, from)) != cudaSuccess) return (int)ce;
        if ((ce = cudaStreamWaitEvent(to, e, 0)) != cudaSuccess) return (int)ce;
        return 0;
    }
};
static thread_local Pipe g_pipe;


// One call: `batch` matrices, workspace carved for pl.per * pl.nslot matrices.  The callbacks get
// (b0 = first matrix of the sub-chunk in the batch, nk = its size, s0 = first workspace record of
// its slot, stream):
//   stageT  enqueues the first stage (it calls stage_T with ws_slice(ws, M, s0, l0))
//   stageQA enqueues QL and apply (w / V / info of the sub-chunk are the caller's business: batch-
//           indexed for the EVD, slot-indexed for the analysis)
//   post    whatever follows (analysis epilogue, read-back hooks)
template <class FT, class FQ, class FA, class FP>
static int run_pipeline(const Plan& pl, int batch, cudaStream_t st, FT stageT, FQ stageQL, FA stageAP, FP post)
{
    if (!pl.pipelined) {
        for (int b0 = 0; b0 < batch; b0 += pl.per) {
            const int nk = (batch - b0 < pl.per) ? batch - b0 : pl.per;
            int rc;
            if ((rc = stageT(b0, nk, 0, 0, st))) return rc;
            if ((rc = stageQL(b0, nk, 0, 0, st, false))) return rc;
            if (pl.ql_mode == QL_CLASSIFY && (rc = stageQL(b0, nk, 0, 0, st, true))) return rc;
            if ((rc = stageAP(b0, nk, 0, 0, st))) return rc;
            if ((rc = post(b0, nk, 0, 0, st))) return rc;
        }
        return 0;
    }
    Pipe& P = g_pipe;
    int rc = P.init();
    if (rc) return rc;
    P.used = 0;
    // every private stream is joined back into `st` on EVERY exit, so that a caller (and the
    // stream-ordered free of an owned workspace) never runs ahead of work still in flight
    auto join_all = [&]() {
        int jr = 0, r2;
        for (int k = 0; k < NT_STREAMS; ++k) if ((r2 = P.link(P.sT[k], st)) && !jr) jr = r2;
        for (int k = 0; k < NA_STREAMS; ++k) if ((r2 = P.link(P.sA[k], st)) && !jr) jr = r2;
        for (int k = 0; k < NQ_STREAMS; ++k) if ((r2 = P.link(P.sQ[k], st)) && !jr) jr = r2;
        return jr;
    };
    for (int k = 0; k < NT_STREAMS && !rc; ++k) rc = P.link(st, P.sT[k]);
    for (int k = 0; k < NA_STREAMS && !rc; ++k) rc = P.link(st, P.sA[k]);
    for (int k = 0; k < NQ_STREAMS && !rc; ++k) rc = P.link(st, P.sQ[k]);
    std::vector<cudaEvent_t> done((size_t)pl.nsub, nullptr);
    for (int k = 0, b0 = 0; b0 < batch && !rc; ++k, b0 += pl.per) {
        const int nk = (batch - b0 < pl.per) ? batch - b0 : pl.per;
        const int s0 = (k % pl.nslot) * pl.per, l0 = (k % pl.nlog) * pl.per;
        cudaStream_t sT = P.sT[k % NT_STREAMS], sQ = P.sQ[k % NQ_STREAMS], sA = P.sA[k % NA_STREAMS];
        if (k >= pl.nslot) {                       // the slot is free when its previous tenant's last kernel is done
            cudaError_t ce = cudaStreamWaitEvent(sT, done[k - pl.nslot], 0);
            if (ce != cudaSuccess) { rc = (int)ce; break; }
        }
        if ((rc = stageT(b0, nk, s0, l0, sT))) break;
        if ((rc = P.link(sT, sQ))) break;
        // (the classifying QL kernel logs nothing: the log slot is only needed by the kernel behind it)
        if (pl.ql_mode == QL_CLASSIFY && (rc = stageQL(b0, nk, s0, l0, sQ, false))) break;
        if (k >= pl.nlog) {                        // ... and so is the log slot
            cudaError_t ce = cudaStreamWaitEvent(sQ, done[k - pl.nlog], 0);
            if (ce != cudaSuccess) { rc = (int)ce; break; }
        }
        if ((rc = stageQL(b0, nk, s0, l0, sQ, pl.ql_mode == QL_CLASSIFY))) break;
        if ((rc = P.link(sQ, sA))) break;
        if ((rc = stageAP(b0, nk, s0, l0, sA))) break;
        if ((rc = post(b0, nk, s0, l0, sA))) break;
        done[k] = P.event();
        if (!done[k]) { rc = (int)cudaErrorMemoryAllocation; break; }
        cudaError_t ce = cudaEventRecord(done[k], sA);
        if (ce != cudaSuccess) { rc = (int)ce; break; }
    }
    const int jr = join_all();
    return rc ? rc : jr;
}

struct ScopedWork {
    void* ptr = nullptr;
    bool owned = false;
    cudaStream_t st = nullptr;
    int acquire(void* user, size_t user_bytes, size_t need, cudaStream_t s, int argpos)
    {
        st = s;
        if (user) {
            if (user_bytes < need || misaligned(user)) return -argpos;
            ptr = user;
            return 0;
        }
        if (need == 0) return 0;
        cudaError_t ce = cudaMallocAsync(&ptr, need, s);
        if (ce != cudaSuccess) return (int)ce;
        owned = true;
        return 0;
    }
    ~ScopedWork() { if (owned && ptr) cudaFreeAsync(ptr, st); }
};

// ---- fp32 variant -----------------------------------------------------
template <int MT>
static int f32_tridiag_run(const float* A, Workspace ws, int M, int n, cudaStream_t st)
{
    const size_t smem = fast_tridiag_smem<MT, float>();
    cudaError_t ce;
    if constexpr (MT == 64) {
        if (t_opt.split && M > 48) {
            if ((ce = allow_smem(fast_tridiag<MT, false, false, float, true>, smem)) != cudaSuccess) return (int)ce;
            KLAUNCH("fast_tridiag_head<f32>", st,
                    (fast_tridiag<MT, false, false, float, true><<<n, FastCfg<MT>::NT, smem, st>>>(
                        A, static_cast<float*>(nullptr), ws, M, nullptr, nullptr, nullptr, 0, 0.0, nullptr, GridArgs{}, n)));
            KLAUNCH("fast_tridiag_tail<f32>", st, fast_tridiag_tail<float><<<n, 32, fast_tridiag_tail_smem<float>(), st>>>(ws, M));
            return 0;
        }
    }
    if constexpr (MT == 64 || MT == 48) {
        if (t_opt.pair > 0) {
            const size_t ps = fast_tridiag_smem_pair<MT, float, true>();
            if ((ce = allow_smem(fast_tridiag<MT, false, false, float, false, true>, ps)) != cudaSuccess) return (int)ce;
            KLAUNCH("fast_tridiag<f32>", st,
                    (fast_tridiag<MT, false, false, float, false, true><<<(n + 1) / 2, FastCfg<MT>::NT, ps, st>>>(
                        A, static_cast<float*>(nullptr), ws, M, nullptr, nullptr, nullptr, 0, 0.0, nullptr, GridArgs{}, n)));
            return 0;
        }
    }
    if ((ce = allow_smem(fast_tridiag<MT, false, false, float>, smem)) != cudaSuccess) return (int)ce;
    KLAUNCH("fast_tridiag<f32>", st,
            fast_tridiag<MT, false, false, float><<<n, FastCfg<MT>::NT, smem, st>>>(
                A, static_cast<float*>(nullptr), ws, M, nullptr, nullptr, nullptr, 0, 0.0, nullptr, GridArgs{}, n));
    return 0;
}
template <int MT>
static int f32_apply_run(float* V, double* wd, float* w, int* info, Workspace ws, int M, int n, cudaStream_t st)
{
    const size_t smem = fast_apply_f32_smem<MT>(ws.swcap);
    cudaError_t ce;
    if ((ce = allow_smem(fast_apply_f32<MT>, smem)) != cudaSuccess) return (int)ce;
    KLAUNCH("fast_apply<f32>", st, fast_apply_f32<MT><<<n, FastCfg<MT>::NT, smem, st>>>(V, wd, w, info, ws, M));
    return 0;
}

}  // namespace letkf

using namespace letkf;

extern "C" {

// Hooks of the host-buffer entry points: pre(b0, nk, s) is enqueued on the stream of a sub-chunk's
// first kernel before it (wait for the sub-chunk's inputs), post(b0, nk, s) after its last kernel
// (start the read-back).  b0 counts from the start of the (device) call.
struct PassHooks {
    int (*pre)(void* ctx, int b0, int nk, cudaStream_t s);
    int (*post)(void* ctx, int b0, int nk, cudaStream_t s);
    void* ctx;
};
static thread_local const PassHooks* t_hooks = nullptr;   // set by the host entry points only

static size_t syev_need(int M, const Plan& pl) { return plan_bytes(M, (size_t)pl.per * pl.nslot, (size_t)pl.per * pl.nlog, 0, pl.two_pass); }

size_t letkf_syev_workspace_bytes(int M, int batch)
{
    EntryScope scope;
    if (M < 1 || M > LETKF_MAX_M || batch < 1) return 0;
    return syev_need(M, make_plan(M, batch, 0, 0));
}

// the EVD of `batch` matrices on device buffers, workspace at `base` (carved per `pl`)
static int syev_core(const double* A, int M, int batch, double* w, double* V, int* info, void* base,
                     const Plan& pl, cudaStream_t st)
{
    Workspace ws;
    carve(ws, base, M, pl.per * pl.nslot, pl.per * pl.nlog, pl.two_pass);
    const PassHooks* hooks = t_hooks;
    auto stageT = [&](int b0, int nk, int s0, int l0, cudaStream_t s) {
        if (hooks) { const int rc = hooks->pre(hooks->ctx, b0, nk, s); if (rc) return rc; }
        return stage_T(A + (size_t)b0 * M * M, M, nk, V + (size_t)b0 * M * M, ws_slice(ws, M, s0, l0), s, nullptr);
    };
    auto stageQL = [&](int b0, int nk, int s0, int l0, cudaStream_t s, bool logpass) {
        if (logpass) return stage_QLlog(M, nk, w + (size_t)b0 * M, info ? info + b0 : nullptr, ws_slice(ws, M, s0, l0), s, pl.bisect);
        if (pl.bisect) return stage_bisect(M, nk, w + (size_t)b0 * M, info ? info + b0 : nullptr, ws_slice(ws, M, s0, l0), s);
        return stage_QL(M, nk, w + (size_t)b0 * M, info ? info + b0 : nullptr, ws_slice(ws, M, s0, l0), s, pl.ql_mode);
    };
    auto stageAP = [&](int b0, int nk, int s0, int l0, cudaStream_t s) {
        return stage_AP(M, nk, w + (size_t)b0 * M, V + (size_t)b0 * M * M, info ? info + b0 : nullptr, ws_slice(ws, M, s0, l0), s);
    };
    auto post = [&](int b0, int nk, int, int, cudaStream_t s) { return hooks ? hooks->post(hooks->ctx, b0, nk, s) : 0; };
    return run_pipeline(pl, batch, st, stageT, stageQL, stageAP, post);
}

int letkf_syev_batched(const double* A, int M, int batch, double* w, double* V, int* info,
                       void* work, size_t work_bytes, void* stream)
{
    EntryScope scope;
    g_launches = 0;
    if (M < 1 || M > LETKF_MAX_M) return -2;
    if (batch < 0) return -3;
    if (batch == 0) return LETKF_OK;
    if (!A || misaligned(A)) return -1;
    if (!w || misaligned(w)) return -4;
    if (!V || misaligned(V)) return -5;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    prof_reset(st);
    const Plan pl = make_plan(M, batch, 0, work ? work_bytes : 0);
    ScopedWork sw;
    int rc = sw.acquire(work, work_bytes, syev_need(M, pl), st, 7);
    if (rc) return rc;
    return syev_core(A, M, batch, w, V, info, sw.ptr, pl, st);
}

// ---- the entry point that allocates nothing (letkf.h: letkf_syev_batched_static) ---------------------
// The kernels' scratch memory is this file-scope array: one per GPU that loads the library, held
// until exit.  In host code `g_static_work` is only a stand-in for the symbol, not a device address:
// the address is looked up once per device (with that device current) and cached here.
static __device__ __align__(256) unsigned char g_static_work[LETKF_STATIC_WORK_BYTES];
static const int STATIC_MAX_DEVICES = 64;
static void* g_static_ptr[STATIC_MAX_DEVICES] = {};
static std::mutex g_static_mu;

static int static_work_ptr(void** out)
{
    int dev = 0;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce != cudaSuccess) return (int)ce;
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return (int)cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        if ((ce = cudaGetSymbolAddress(&p, g_static_work)) != cudaSuccess) return (int)ce;
        if (!p || misaligned(p)) return (int)cudaErrorInvalidSymbol;
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return 0;
}

// one chunk of `batch` matrices on the caller's stream: the plan letkf_syev_batched takes when it does not pipeline
static Plan static_plan(int M, int batch)
{
    Plan pl = make_plan(M, batch, 0, 0);
    pl.per = batch; pl.nslot = 1; pl.nlog = 1; pl.nsub = 1; pl.pipelined = false;
    return pl;
}

int letkf_syev_static_max_batch(int M)
{
    EntryScope scope;
    if (M < 1 || M > LETKF_MAX_M) return 0;
    int lo = 0, hi = 1 << 20;                  // largest batch whose workspace fits (the size grows with the batch wherever it fits)
    while (lo < hi) {
        const int mid = lo + (hi - lo + 1) / 2;
        if (syev_need(M, static_plan(M, mid)) <= (size_t)LETKF_STATIC_WORK_BYTES) lo = mid; else hi = mid - 1;
    }
    return lo;
}

int letkf_syev_batched_static(const double* A, int M, int batch, double* w, double* V, int* info, void* stream)
{
    EntryScope scope;
    g_launches = 0;
    if (M < 1 || M > LETKF_MAX_M) return -2;
    if (batch < 0) return -3;
    if (batch == 0) return LETKF_OK;
    if (!A || misaligned(A)) return -1;
    if (!w || misaligned(w)) return -4;
    if (!V || misaligned(V)) return -5;
    const Plan pl = static_plan(M, batch);
    if (syev_need(M, pl) > (size_t)LETKF_STATIC_WORK_BYTES) return LETKF_ERR_STATIC_CAPACITY;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    void* base = nullptr;
    int rc = static_work_ptr(&base);
    if (rc) return rc;
    struct ProfOff {                           // the profiling aid creates events and a counter: not here
        bool was = g_prof.on;
        ProfOff() { g_prof.on = false; }
        ~ProfOff() { g_prof.on = was; }
    } prof_off;
    Workspace ws;
    carve(ws, base, M, batch, batch, pl.two_pass);
    // the array keeps the last call's contents: the records a matrix starts from are cleared
    cudaError_t ce;
    if ((ce = cudaMemsetAsync(ws.flags, 0, sizeof(int) * (size_t)batch, st)) != cudaSuccess) return (int)ce;
    if ((ce = cudaMemsetAsync(ws.nsweeps, 0, sizeof(int) * (size_t)batch, st)) != cudaSuccess) return (int)ce;
    return syev_core(A, M, batch, w, V, info, base, pl, st);
}

size_t letkf_syev_f32_workspace_bytes(int M, int batch)
{
    EntryScope scope;
    if (M < 1 || M > 64 || batch < 1) return 0;
    t_opt.qform = 0; t_opt.force_generic = 0;
    const size_t extra = sizeof(double) * (size_t)M;
    const Plan pl = make_plan(M, batch, extra, 0);
    return plan_bytes(M, (size_t)pl.per * pl.nslot, (size_t)pl.per * pl.nlog, extra, pl.two_pass);
}

int letkf_syev_batched_f32(const float* A, int M, int batch, float* w, float* V, int* info,
                           void* work, size_t work_bytes, void* stream)
{
    EntryScope scope;
    g_launches = 0;
    if (M < 1 || M > 64) return -2;            // the register path only (the paper's Table I sizes)
    if (batch < 0) return -3;
    if (batch == 0) return LETKF_OK;
    if (!A || misaligned(A)) return -1;
    if (!w || misaligned(w)) return -4;
    if (!V || misaligned(V)) return -5;
    t_opt.qform = 0; t_opt.force_generic = 0;  // this entry point has the reflector form only
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    prof_reset(st);
    const size_t extra = sizeof(double) * (size_t)M;
    const Plan pl = make_plan(M, batch, extra, work ? work_bytes : 0);
    ScopedWork sw;
    int rc = sw.acquire(work, work_bytes, plan_bytes(M, (size_t)pl.per * pl.nslot, (size_t)pl.per * pl.nlog, extra, pl.two_pass), st, 7);
    if (rc) return rc;
    Workspace ws;
    const size_t off = carve(ws, sw.ptr, M, pl.per * pl.nslot, pl.per * pl.nlog, pl.two_pass);
    double* wd = reinterpret_cast<double*>(reinterpret_cast<char*>(sw.ptr) + off);      // [slot matrices][M] eigenvalues in fp64
    if (M == 1) {      // nothing to reduce: w = A, V = 1 (the kernels want M >= 2)
        KLAUNCH("f32_order_one", st, f32_order_one<<<(batch + 255) / 256, 256, 0, st>>>(A, w, V, info, batch));
        return LETKF_OK;
    }
    auto stageT = [&](int b0, int nk, int s0, int l0, cudaStream_t s) {
        const Workspace wk = ws_slice(ws, M, s0, l0);
        switch (fast_bucket(M)) {
            case 16: return f32_tridiag_run<16>(A + (size_t)b0 * M * M, wk, M, nk, s);
            case 32: return f32_tridiag_run<32>(A + (size_t)b0 * M * M, wk, M, nk, s);
            case 48: return f32_tridiag_run<48>(A + (size_t)b0 * M * M, wk, M, nk, s);
            default: return f32_tridiag_run<64>(A + (size_t)b0 * M * M, wk, M, nk, s);
        }
    };
    auto stageQL = [&](int b0, int nk, int s0, int l0, cudaStream_t s, bool logpass) {
        const Workspace wk = ws_slice(ws, M, s0, l0);
        int* ik = info ? info + b0 : nullptr;
        if (logpass) return stage_QLlog(M, nk, wd + (size_t)s0 * M, ik, wk, s, pl.bisect);
        if (pl.bisect) return stage_bisect(M, nk, wd + (size_t)s0 * M, ik, wk, s);
        return stage_QL(M, nk, wd + (size_t)s0 * M, ik, wk, s, pl.ql_mode);
    };
    auto stageAP = [&](int b0, int nk, int s0, int l0, cudaStream_t s) {
        const Workspace wk = ws_slice(ws, M, s0, l0);
        int* ik = info ? info + b0 : nullptr;
        float* Vk = V + (size_t)b0 * M * M;
        float* wk_ = w + (size_t)b0 * M;
        switch (fast_bucket(M)) {
            case 16: return f32_apply_run<16>(Vk, wd + (size_t)s0 * M, wk_, ik, wk, M, nk, s);
            case 32: return f32_apply_run<32>(Vk, wd + (size_t)s0 * M, wk_, ik, wk, M, nk, s);
            case 48: return f32_apply_run<48>(Vk, wd + (size_t)s0 * M, wk_, ik, wk, M, nk, s);
            default: return f32_apply_run<64>(Vk, wd + (size_t)s0 * M, wk_, ik, wk, M, nk, s);
        }
    };
    auto post = [&](int, int, int, int, cudaStream_t) { return 0; };
    return run_pipeline(pl, batch, st, stageT, stageQL, stageAP, post);
}

// per-matrix bytes the analysis keeps per slot beside the EVD workspace: Q / V (not on the fused
// M <= 64 path, where V never leaves the SM), lam, g
static size_t analysis_extra(int M, bool keepV) { return sizeof(double) * ((keepV ? (size_t)M * M : 0) + 2 * (size_t)M); }
static bool analysis_fused(int M, int nstate, bool wantW) { return !wantW && use_fast(M) && nstate <= EPI_NS_MAX; }
// is a Q / V buffer needed per slot?  (not when a6-a9 are fused into fast_apply and Q is never formed)
static bool analysis_keepV(int M, int nstate, bool wantW) { return !analysis_fused(M, nstate, wantW) || t_opt.qform; }
static size_t analysis_need(int M, const Plan& pl, size_t extra) { return plan_bytes(M, (size_t)pl.per * pl.nslot, (size_t)pl.per * pl.nlog, extra, pl.two_pass); }

size_t letkf_analysis_workspace_bytes(int M, int p, int nstate, int batch)
{
    EntryScope scope;
    (void)p; (void)nstate;
    if (M < 1 || M > LETKF_MAX_M || batch < 1) return 0;
    // sized for the form that needs most (W requested: V is kept per slot)
    const size_t extra = analysis_extra(M, true);
    return analysis_need(M, make_plan(M, batch, extra, 0), extra);
}

// does the grid form run with the gather fused into the tridiagonalisation kernel?
static bool grid_fused(int M, int nstate) { return use_fast(M) && nstate <= EPI_NS_MAX; }

static size_t grid_extra(int M, int p, int nstate)
{
    size_t e = analysis_extra(M, true);
    if (!grid_fused(M, nstate)) e += sizeof(double) * ((size_t)p * M + 2 * (size_t)p);      // materialised Y_loc, d, r
    return e;
}

size_t letkf_analysis_grid_workspace_bytes(int M, int V, int Ny, int Nx, int hw, int nstate)
{
    EntryScope scope;
    if (M < 2 || M > LETKF_MAX_M || V < 1 || Ny < 1 || Nx < 1 || hw < 0 || nstate < 1) return 0;
    const long npts = (long)Ny * Nx;
    if (npts > 0x7fffffffL) return 0;
    const int batch = (int)npts, p = V * (2 * hw + 1) * (2 * hw + 1);
    const size_t extra = grid_extra(M, p, nstate);
    return analysis_need(M, make_plan(M, batch, extra, 0), extra) + align_up(sizeof(double) * (size_t)V * npts, 256) + 4 * 256;
}

// a1-a9 for `batch` grid points.  Either (Yb, d, rinv_loc) or `grid` (local observations gathered
// from the fields: inside the tridiagonalisation kernel when grid_fused(), else materialised per
// slot in the workspace).  `work` holds analysis_need(M, pl, extra) bytes.
static int analysis_core(const double* Yb, const double* d, const double* rinv_loc, const GridArgs* grid,
                         const double* Xb, int M, int p, int nstate, int batch, double rho,
                         double* Xa, double* W, double* wbar, int* info,
                         void* work, const Plan& pl, size_t extra, cudaStream_t st)
{
    (void)extra;
    const int nrec = pl.per * pl.nslot;
    Workspace ws;
    size_t off = carve(ws, work, M, nrec, pl.per * pl.nlog, pl.two_pass);
    char* base = reinterpret_cast<char*>(work);
    const bool fused = analysis_fused(M, nstate, W != nullptr);
    const bool fuse_gather = grid && !W && grid_fused(M, nstate);
    double* Vbuf = nullptr;
    if (analysis_keepV(M, nstate, W != nullptr)) { Vbuf = reinterpret_cast<double*>(base + off); off += align_up(sizeof(double) * (size_t)M * M * nrec, 256); }
    double* lam  = reinterpret_cast<double*>(base + off); off += align_up(sizeof(double) * (size_t)M * nrec, 256);
    double* gbuf = reinterpret_cast<double*>(base + off); off += align_up(sizeof(double) * (size_t)M * nrec, 256);
    double *gYb = nullptr, *gd = nullptr, *gr = nullptr;
    if (grid && !fuse_gather) {
        gYb = reinterpret_cast<double*>(base + off); off += align_up(sizeof(double) * (size_t)p * M * nrec, 256);
        gd = reinterpret_cast<double*>(base + off);  off += align_up(sizeof(double) * (size_t)p * nrec, 256);
        gr = reinterpret_cast<double*>(base + off);  off += align_up(sizeof(double) * (size_t)p * nrec, 256);
    }

    const double shift = (double)(M - 1) / rho;
    cudaError_t ce;
    const size_t ep_smem = sizeof(double) * (3 * (size_t)M + 2 * (size_t)nstate + 2 * (size_t)nstate * M);
    if (ep_smem > 200 * 1024) return -7;
    auto epi_kernel = [&](bool wantW) {
        const int ks = (M + 31) / 32;
        if (wantW) return ks <= 2 ? generic_epilogue<true, 2> : (ks <= 4 ? generic_epilogue<true, 4> : (ks <= 6 ? generic_epilogue<true, 6> : generic_epilogue<true, 8>));
        return ks <= 2 ? generic_epilogue<false, 2> : (ks <= 4 ? generic_epilogue<false, 4> : (ks <= 6 ? generic_epilogue<false, 6> : generic_epilogue<false, 8>));
    };
    auto epi = epi_kernel(W != nullptr);
    if ((ce = allow_smem(epi, ep_smem)) != cudaSuccess) return (int)ce;
    const PassHooks* hooks = t_hooks;

    auto stageT = [&](int b0, int nk, int s0, int l0, cudaStream_t s) {
        if (hooks) { const int hrc = hooks->pre(hooks->ctx, b0, nk, s); if (hrc) return hrc; }
        GramArgs ga{nullptr, nullptr, nullptr, p, shift, gbuf + (size_t)s0 * M, GridArgs{}};
        if (grid) {
            GridArgs gk = *grid;
            gk.point0 = grid->point0 + b0;
            if (fuse_gather) {
                ga.grid = gk;
            } else {
                KLAUNCH("grid_gather", s,
                        grid_gather<<<nk, 256, 0, s>>>(gk, M, p, gYb + (size_t)s0 * p * M, gd + (size_t)s0 * p, gr + (size_t)s0 * p));
                ga.Yb = gYb + (size_t)s0 * p * M; ga.d = gd + (size_t)s0 * p; ga.r = gr + (size_t)s0 * p;
            }
        } else {
            ga.Yb = Yb + (size_t)b0 * p * M; ga.d = d + (size_t)b0 * p; ga.r = rinv_loc + (size_t)b0 * p;
        }
        double* Vk = Vbuf ? Vbuf + (size_t)s0 * M * M : nullptr;
        return stage_T(Vk, M, nk, Vk, ws_slice(ws, M, s0, l0), s, &ga);
    };
    auto stageQL = [&](int b0, int nk, int s0, int l0, cudaStream_t s, bool logpass) {
        if (logpass) return stage_QLlog(M, nk, lam + (size_t)s0 * M, info ? info + b0 : nullptr, ws_slice(ws, M, s0, l0), s, pl.bisect);
        if (pl.bisect) return stage_bisect(M, nk, lam + (size_t)s0 * M, info ? info + b0 : nullptr, ws_slice(ws, M, s0, l0), s);
        return stage_QL(M, nk, lam + (size_t)s0 * M, info ? info + b0 : nullptr, ws_slice(ws, M, s0, l0), s, pl.ql_mode);
    };
    // a6-a9: fused into fast_apply when W is not wanted (V then never leaves the SM); the any-M
    // kernel otherwise
    auto stageAP = [&](int b0, int nk, int s0, int l0, cudaStream_t s) {
        EpiArgs ep{lam + (size_t)s0 * M, gbuf + (size_t)s0 * M, Xb + (size_t)b0 * nstate * M, Xa + (size_t)b0 * nstate * M,
                   wbar ? wbar + (size_t)b0 * M : nullptr, nstate};
        return stage_AP(M, nk, lam + (size_t)s0 * M, Vbuf ? Vbuf + (size_t)s0 * M * M : nullptr, info ? info + b0 : nullptr,
                        ws_slice(ws, M, s0, l0), s, fused ? &ep : nullptr);
    };
    auto post = [&](int b0, int nk, int s0, int l0, cudaStream_t s) -> int {
        if (!fused) {
            KLAUNCH("generic_epilogue", s,
                    epi<<<nk, 256, ep_smem, s>>>(
                        Vbuf + (size_t)s0 * M * M, lam + (size_t)s0 * M, gbuf + (size_t)s0 * M,
                        Xb + (size_t)b0 * nstate * M, M, nstate, nk, Xa + (size_t)b0 * nstate * M,
                        W ? W + (size_t)b0 * M * M : nullptr, wbar ? wbar + (size_t)b0 * M : nullptr, nullptr));
        }
        return hooks ? hooks->post(hooks->ctx, b0, nk, s) : 0;
    };
    return run_pipeline(pl, batch, st, stageT, stageQL, stageAP, post);
}

int letkf_analysis_batched(const double* Yb, const double* d, const double* rinv_loc,
                           const double* Xb, int M, int p, int nstate, int batch, double rho,
                           double* Xa, double* W, double* wbar, int* info,
                           void* work, size_t work_bytes, void* stream)
{
    EntryScope scope;
    g_launches = 0;
    if (M < 2 || M > LETKF_MAX_M) return -5;   // M = 1 has no ensemble spread: Eq.15 is 0/0
    if (p < 0) return -6;
    if (nstate < 1) return -7;
    if (batch < 0) return -8;
    if (!(rho > 0.0)) return -9;
    if (batch == 0) return LETKF_OK;
    if (p > 0 && (!Yb || misaligned(Yb))) return -1;
    if (p > 0 && (!d || misaligned(d))) return -2;
    if (p > 0 && (!rinv_loc || misaligned(rinv_loc))) return -3;
    if (!Xb || misaligned(Xb)) return -4;
    if (!Xa || misaligned(Xa)) return -10;
    if (W && misaligned(W)) return -11;
    if (wbar && misaligned(wbar)) return -12;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    prof_reset(st);
    const size_t extra = analysis_extra(M, analysis_keepV(M, nstate, W != nullptr));
    const Plan pl = make_plan(M, batch, extra, work ? work_bytes : 0);
    ScopedWork sw;
    int rc = sw.acquire(work, work_bytes, analysis_need(M, pl, extra), st, 14);
    if (rc) return rc;
    return analysis_core(Yb, d, rinv_loc, nullptr, Xb, M, p, nstate, batch, rho, Xa, W, wbar, info, sw.ptr, pl, extra, st);
}

int letkf_analysis_batched_evdfree(const double* Yb, const double* d, const double* rinv_loc,
                                   const double* Xb, int M, int p, int nstate, int batch, double rho,
                                   double* Xa, double* W, double* wbar, int* info, void* stream)
{
    EntryScope scope;
    g_launches = 0;
    if (M < 2 || M > NS_MT) return -5;
    if (p < 0) return -6;
    if (nstate < 1 || nstate > 16) return -7;
    if (batch < 0) return -8;
    if (!(rho > 0.0)) return -9;
    if (batch == 0) return LETKF_OK;
    if (p > 0 && (!Yb || misaligned(Yb))) return -1;
    if (p > 0 && (!d || misaligned(d))) return -2;
    if (p > 0 && (!rinv_loc || misaligned(rinv_loc))) return -3;
    if (!Xb || misaligned(Xb)) return -4;
    if (!Xa || misaligned(Xa)) return -10;
    if (W && misaligned(W)) return -11;
    if (wbar && misaligned(wbar)) return -12;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    prof_reset(st);
    cudaError_t ce;
    if ((ce = allow_smem(ns_analysis_kernel, NS_SMEM)) != cudaSuccess) return (int)ce;
    KLAUNCH("ns_analysis_kernel", st,
            ns_analysis_kernel<<<batch, NS_NT, NS_SMEM, st>>>(Yb, d, rinv_loc, Xb, M, p, nstate, rho, Xa, W, wbar, info));
    return LETKF_OK;
}

int letkf_analysis_grid(const double* Yf, const double* yo, const unsigned char* obs_mask, const double* Xb,
                        int M, int V, int Ny, int Nx, int nstate, int hw, int loc_kind, double loc_scale,
                        double sigma_o, double rho, double* Xa, double* wbar, int* info,
                        void* work, size_t work_bytes, void* stream)
{
    EntryScope scope;
    g_launches = 0;
    if (M < 2 || M > LETKF_MAX_M) return -5;
    if (V < 1) return -6;
    if (Ny < 1) return -7;
    if (Nx < 1 || (long)Ny * Nx > 0x7fffffffL) return -8;
    if (nstate < 1) return -9;
    if (hw < 0) return -10;
    if (loc_kind != 0 && loc_kind != 1) return -11;
    if (!(loc_scale > 0.0)) return -12;
    if (!(sigma_o > 0.0)) return -13;
    if (!(rho > 0.0)) return -14;
    if (!Yf || misaligned(Yf)) return -1;
    if (!yo || misaligned(yo)) return -2;
    if (!Xb || misaligned(Xb)) return -4;
    if (!Xa || misaligned(Xa)) return -15;
    if (wbar && misaligned(wbar)) return -16;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    prof_reset(st);
    const int batch = Ny * Nx, side = 2 * hw + 1, p = V * side * side;
    // carve: [ybar][analysis workspace (with the materialised Y_loc of the slots when the gather is not fused)]
    const size_t ybytes = align_up(sizeof(double) * (size_t)V * batch, 256);
    const size_t extra = grid_extra(M, p, nstate) - (analysis_keepV(M, nstate, false) ? 0 : sizeof(double) * (size_t)M * M);
    const Plan pl = make_plan(M, batch, extra, work ? (work_bytes > ybytes ? work_bytes - ybytes : 1) : 0);
    ScopedWork sw;
    int rc = sw.acquire(work, work_bytes, ybytes + analysis_need(M, pl, extra), st, 18);
    if (rc) return rc;
    char* base = reinterpret_cast<char*>(sw.ptr);
    double* ybar = reinterpret_cast<double*>(base);
    const long nobs = (long)V * batch;
    KLAUNCH("grid_obs_mean", st, grid_obs_mean<<<(unsigned)((nobs + 7) / 8), 256, 0, st>>>(Yf, ybar, nobs, M));
    GridArgs g{Yf, ybar, yo, obs_mask, V, Ny, Nx, hw, loc_kind, loc_scale, 1.0 / (sigma_o * sigma_o), 0};
    return analysis_core(nullptr, nullptr, nullptr, &g, Xb, M, p, nstate, batch, rho,
                         Xa, nullptr, wbar, info, base + ybytes, pl, extra, st);
}

// ---- host-buffer entry points -----------------------------------------------------------------
// A pass of the batch lives on the device at a time; the sub-chunks of the kernel pipeline are
// copied in one after the other on a copy-in stream, each sub-chunk's first kernel waits for its
// own copy only, and its read-back starts on a copy-out stream as soon as its last kernel is done:
// both copy engines and the SMs overlap (PCIe is full duplex).  The device staging arena is kept by
// the calling host thread between calls (letkf_host_release() frees it); the call returns after the
// last byte has reached the host.
struct HostPipe {
    int dev = -1;
    cudaStream_t s[2] = {nullptr, nullptr};
    cudaStream_t sC = nullptr;    // the stream the kernels of a host call are forked from
    std::vector<cudaEvent_t> ev;
    int events(size_t n)
    {
        while (ev.size() < n) {
            cudaEvent_t e;
            cudaError_t ce = cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
            if (ce != cudaSuccess) return (int)ce;
            ev.push_back(e);
        }
        return 0;
    }
    char* arena = nullptr;        // device staging memory, grown on demand and kept between calls
    size_t arena_bytes = 0;       // (re-allocating > 1 GB per call costs more than the whole EVD)
    int reserve(size_t bytes)
    {
        if (bytes <= arena_bytes) return 0;
        release();
        cudaError_t ce = cudaMalloc(reinterpret_cast<void**>(&arena), bytes);
        if (ce != cudaSuccess) { arena = nullptr; return (int)ce; }
        arena_bytes = bytes;
        return 0;
    }
    void release()
    {
        if (arena) cudaFree(arena);
        arena = nullptr;
        arena_bytes = 0;
    }
    int init()
    {
        int d = 0;
        cudaError_t ce = cudaGetDevice(&d);
        if (ce != cudaSuccess) return (int)ce;
        if (d == dev) return 0;
        if (dev >= 0) {                      // the thread moved to another device: free what lives on the old one
            cudaSetDevice(dev);
            release();
            for (auto& x : s) if (x) { cudaStreamDestroy(x); x = nullptr; }
            if (sC) { cudaStreamDestroy(sC); sC = nullptr; }
            for (auto e : ev) cudaEventDestroy(e);
            ev.clear();
            cudaSetDevice(d);
        }
        for (int k = 0; k < 2; ++k)
            if ((ce = cudaStreamCreateWithFlags(&s[k], cudaStreamNonBlocking)) != cudaSuccess) return (int)ce;
        if ((ce = cudaStreamCreateWithFlags(&sC, cudaStreamNonBlocking)) != cudaSuccess) return (int)ce;
        dev = d;
        return 0;
    }
    // everything of a pass must have left the arena before it is reused or the call returns
    int drain()
    {
        cudaError_t e0 = cudaStreamSynchronize(sC), e1 = cudaStreamSynchronize(s[1]), e2 = cudaStreamSynchronize(s[0]);
        return (int)(e0 != cudaSuccess ? e0 : (e1 != cudaSuccess ? e1 : e2));
    }
};
static thread_local HostPipe g_hpipe;

#define CUDA_TRY(call) do { cudaError_t ce_ = (call); if (ce_ != cudaSuccess) return (int)ce_; } while (0)

// matrices per pass of a host call: what a staging arena of HOST_ARENA_CAP holds (or the test option)
static const size_t HOST_ARENA_CAP = (size_t)16 << 30;
static int host_pass_size(int batch, size_t bytes_per_matrix)
{
    size_t c = t_opt.host_pass > 0 ? (size_t)t_opt.host_pass : HOST_ARENA_CAP / (bytes_per_matrix ? bytes_per_matrix : 1);
    if (c < 1) c = 1;
    if (c > (size_t)batch) c = (size_t)batch;
    return (int)c;
}

// context of the copy hooks: the inputs of sub-chunk k have arrived when evH[k] fires; the outputs
// listed here (per matrix / grid point: host base, device base, bytes) are read back after its last kernel
struct HostCtx {
    int per, nout;
    char* host[4]; const char* dev[4]; size_t bytes[4];
    cudaStream_t sD;
    const cudaEvent_t* evH;
    const cudaEvent_t* evC;
    void add(void* h, const void* dv, size_t b) { host[nout] = static_cast<char*>(h); dev[nout] = static_cast<const char*>(dv); bytes[nout] = b; ++nout; }
};
static int host_pre(void* c, int b0, int, cudaStream_t s)
{
    HostCtx* x = static_cast<HostCtx*>(c);
    return (int)cudaStreamWaitEvent(s, x->evH[b0 / x->per], 0);
}
static int host_post(void* c, int b0, int nk, cudaStream_t s)
{
    HostCtx* x = static_cast<HostCtx*>(c);
    cudaEvent_t e = x->evC[b0 / x->per];
    CUDA_TRY(cudaEventRecord(e, s));
    CUDA_TRY(cudaStreamWaitEvent(x->sD, e, 0));
    for (int q = 0; q < x->nout; ++q)
        CUDA_TRY(cudaMemcpyAsync(x->host[q] + (size_t)b0 * x->bytes[q], x->dev[q] + (size_t)b0 * x->bytes[q],
                                 x->bytes[q] * (size_t)nk, cudaMemcpyDeviceToHost, x->sD));
    return 0;
}
struct HooksGuard {
    explicit HooksGuard(const PassHooks* h) { t_hooks = h; }
    ~HooksGuard() { t_hooks = nullptr; }
};

int letkf_syev_batched_host(const double* A, int M, int batch, double* w, double* V, int* info)
{
    EntryScope scope;
    g_launches = 0;
    if (M < 1 || M > LETKF_MAX_M) return -2;
    if (batch < 0) return -3;
    if (batch == 0) return LETKF_OK;
    if (!A) return -1;
    if (!w) return -4;
    if (!V) return -5;
    int rc = g_hpipe.init();
    if (rc) return rc;
    const size_t mat = sizeof(double) * (size_t)M * M, vec = sizeof(double) * (size_t)M;
    const int chunk = host_pass_size(batch, mat + vec + sizeof(int));
    const Plan pl = make_plan(M, chunk, 0, 0);
    const size_t wsb = align_up(syev_need(M, pl), 256);
    const size_t oV = 0, ow = align_up(mat * chunk, 256), oi = ow + align_up(vec * chunk, 256);
    const size_t owk = oi + align_up(sizeof(int) * (size_t)chunk, 256);
    if ((rc = g_hpipe.reserve(owk + wsb))) return rc;
    char* base = g_hpipe.arena;
    double* dV = reinterpret_cast<double*>(base + oV);
    double* dw = reinterpret_cast<double*>(base + ow);
    int* dinfo = reinterpret_cast<int*>(base + oi);
    cudaStream_t sH = g_hpipe.s[0], sD = g_hpipe.s[1], sC = g_hpipe.sC;
    int launches = 0;
    for (int b0 = 0; b0 < batch && rc == 0; b0 += chunk) {
        const int n = (batch - b0 < chunk) ? batch - b0 : chunk;
        const Plan pn = (n == chunk) ? pl : make_plan(M, n, 0, wsb);
        prof_reset(sC);
        if ((rc = g_hpipe.events(2 * (size_t)pn.nsub))) break;
        const cudaEvent_t* evH = g_hpipe.ev.data();
        const cudaEvent_t* evC = g_hpipe.ev.data() + pn.nsub;
        for (int k = 0, c0 = 0; c0 < n && rc == 0; ++k, c0 += pn.per) {
            const int nk = (n - c0 < pn.per) ? n - c0 : pn.per;
            cudaError_t ce = cudaMemcpyAsync(dV + (size_t)c0 * M * M, A + (size_t)(b0 + c0) * M * M, mat * nk, cudaMemcpyHostToDevice, sH);
            if (ce == cudaSuccess) ce = cudaEventRecord(evH[k], sH);
            rc = (int)ce;
        }
        if (rc == 0) rc = (int)cudaMemsetAsync(dinfo, 0, sizeof(int) * (size_t)n, sC);
        if (rc == 0) {
            HostCtx ctx{pn.per, 0, {}, {}, {}, sD, evH, evC};
            ctx.add(V + (size_t)b0 * M * M, dV, mat);
            ctx.add(w + (size_t)b0 * M, dw, vec);
            if (info) ctx.add(info + b0, dinfo, sizeof(int));
            PassHooks hooks{host_pre, host_post, &ctx};
            HooksGuard guard(&hooks);
            rc = syev_core(dV, M, n, dw, dV, dinfo, base + owk, pn, sC);     // in place
            launches += g_launches;
        }
        const int dr = g_hpipe.drain();
        if (rc == 0) rc = dr;
    }
    cudaError_t ce = cudaGetLastError();
    if (rc == 0 && ce != cudaSuccess) rc = (int)ce;
    g_launches = launches;
    return rc;
}

int letkf_analysis_batched_host(const double* Yb, const double* d, const double* rinv_loc,
                                const double* Xb, int M, int p, int nstate, int batch, double rho,
                                double* Xa, double* W, double* wbar, int* info)
{
    EntryScope scope;
    g_launches = 0;
    if (M < 2 || M > LETKF_MAX_M) return -5;
    if (p < 0) return -6;
    if (nstate < 1) return -7;
    if (batch < 0) return -8;
    if (!(rho > 0.0)) return -9;
    if (batch == 0) return LETKF_OK;
    if (p > 0 && !Yb) return -1;
    if (p > 0 && !d) return -2;
    if (p > 0 && !rinv_loc) return -3;
    if (!Xb) return -4;
    if (!Xa) return -10;
    int rc = g_hpipe.init();
    if (rc) return rc;
    // as letkf_syev_batched_host: one pass on the device at a time, inputs copied in sub-chunk by
    // sub-chunk, outputs read back as each sub-chunk's last kernel finishes
    const size_t sYb = sizeof(double) * (size_t)p * M, sd = sizeof(double) * (size_t)p;
    const size_t sX = sizeof(double) * (size_t)nstate * M, sW = sizeof(double) * (size_t)M * M;
    const size_t sw = sizeof(double) * (size_t)M;
    const int chunk = host_pass_size(batch, sYb + 2 * sd + sX + (W ? sW : 0) + sw + sizeof(int));
    const size_t extra = analysis_extra(M, analysis_keepV(M, nstate, W != nullptr));
    const Plan pl = make_plan(M, chunk, extra, 0);
    const size_t wsb = align_up(analysis_need(M, pl, extra), 256);
    size_t off[8], total = 0;
    const size_t sizes[8] = {sYb * chunk, sd * chunk, sd * chunk, sX * chunk, W ? sW * chunk : 0,
                             wbar ? sw * chunk : 0, sizeof(int) * (size_t)chunk, wsb};
    for (int k = 0; k < 8; ++k) { off[k] = total; total += align_up(sizes[k] ? sizes[k] : 16, 256); }
    if ((rc = g_hpipe.reserve(total))) return rc;
    char* base = g_hpipe.arena;
    double* dYb = reinterpret_cast<double*>(base + off[0]);
    double* dd = reinterpret_cast<double*>(base + off[1]);
    double* dr = reinterpret_cast<double*>(base + off[2]);
    double* dX = reinterpret_cast<double*>(base + off[3]);
    double* dW = W ? reinterpret_cast<double*>(base + off[4]) : nullptr;
    double* dwb = wbar ? reinterpret_cast<double*>(base + off[5]) : nullptr;
    int* dinfo = reinterpret_cast<int*>(base + off[6]);
    void* dwork = base + off[7];
    cudaStream_t sH = g_hpipe.s[0], sD = g_hpipe.s[1], sC = g_hpipe.sC;
    int launches = 0;
    for (int b0 = 0; b0 < batch && rc == 0; b0 += chunk) {
        const int n = (batch - b0 < chunk) ? batch - b0 : chunk;
        const Plan pn = (n == chunk) ? pl : make_plan(M, n, extra, wsb);
        prof_reset(sC);
        if ((rc = g_hpipe.events(2 * (size_t)pn.nsub))) break;
        const cudaEvent_t* evH = g_hpipe.ev.data();
        const cudaEvent_t* evC = g_hpipe.ev.data() + pn.nsub;
        for (int k = 0, c0 = 0; c0 < n && rc == 0; ++k, c0 += pn.per) {
            const int nk = (n - c0 < pn.per) ? n - c0 : pn.per;
            const size_t g0 = (size_t)(b0 + c0);
            cudaError_t ce = cudaSuccess;
            if (p > 0) {
                ce = cudaMemcpyAsync(dYb + (size_t)c0 * p * M, Yb + g0 * p * M, sYb * nk, cudaMemcpyHostToDevice, sH);
                if (ce == cudaSuccess) ce = cudaMemcpyAsync(dd + (size_t)c0 * p, d + g0 * p, sd * nk, cudaMemcpyHostToDevice, sH);
                if (ce == cudaSuccess) ce = cudaMemcpyAsync(dr + (size_t)c0 * p, rinv_loc + g0 * p, sd * nk, cudaMemcpyHostToDevice, sH);
            }
            if (ce == cudaSuccess) ce = cudaMemcpyAsync(dX + (size_t)c0 * nstate * M, Xb + g0 * nstate * M, sX * nk, cudaMemcpyHostToDevice, sH);
            if (ce == cudaSuccess) ce = cudaEventRecord(evH[k], sH);
            rc = (int)ce;
        }
        if (rc == 0) rc = (int)cudaMemsetAsync(dinfo, 0, sizeof(int) * (size_t)n, sC);
        if (rc == 0) {
            HostCtx ctx{pn.per, 0, {}, {}, {}, sD, evH, evC};
            ctx.add(Xa + (size_t)b0 * nstate * M, dX, sX);
            if (W) ctx.add(W + (size_t)b0 * M * M, dW, sW);
            if (wbar) ctx.add(wbar + (size_t)b0 * M, dwb, sw);
            if (info) ctx.add(info + b0, dinfo, sizeof(int));
            PassHooks hooks{host_pre, host_post, &ctx};
            HooksGuard guard(&hooks);
            rc = analysis_core(dYb, dd, dr, nullptr, dX, M, p, nstate, n, rho, dX, dW, dwb, dinfo, dwork, pn, extra, sC);
            launches += g_launches;
        }
        const int dr_ = g_hpipe.drain();
        if (rc == 0) rc = dr_;
    }
    cudaError_t ce = cudaGetLastError();
    if (rc == 0 && ce != cudaSuccess) rc = (int)ce;
    g_launches = launches;
    return rc;
}

void letkf_host_release(void) { g_hpipe.release(); }

int letkf_analysis_grid_host(const double* Yf, const double* yo, const unsigned char* obs_mask,
                             const double* Xb, int M, int V, int Ny, int Nx, int nstate, int hw,
                             int loc_kind, double loc_scale, double sigma_o, double rho,
                             double* Xa, double* wbar, int* info)
{
    EntryScope scope;
    g_launches = 0;
    if (M < 2 || M > LETKF_MAX_M) return -5;
    if (V < 1) return -6;
    if (Ny < 1) return -7;
    if (Nx < 1 || (long)Ny * Nx > 0x7fffffffL) return -8;
    if (nstate < 1) return -9;
    if (hw < 0) return -10;
    if (loc_kind != 0 && loc_kind != 1) return -11;
    if (!(loc_scale > 0.0)) return -12;
    if (!(sigma_o > 0.0)) return -13;
    if (!(rho > 0.0)) return -14;
    if (!Yf) return -1;
    if (!yo) return -2;
    if (!Xb) return -4;
    if (!Xa) return -15;
    int rc = g_hpipe.init();
    if (rc) return rc;
    // The observation fields (V Ny Nx (M+1) doubles: 17 MB at 128 x 128 x 2 x 64) go in first, whole;
    // the background ensemble follows sub-chunk by sub-chunk and the analysis ensemble comes back
    // the same way (hooks as in letkf_analysis_batched_host).  The whole grid is one pass.
    const int batch = Ny * Nx, side = 2 * hw + 1, p = V * side * side;
    const size_t nobs = (size_t)V * batch;
    const size_t sX = sizeof(double) * (size_t)nstate * M, sw = sizeof(double) * (size_t)M;
    const size_t wsb = align_up(letkf_analysis_grid_workspace_bytes(M, V, Ny, Nx, hw, nstate), 256);
    // the sub-chunk size the device call will use with this workspace (same rule, same inputs)
    const size_t ybytes = align_up(sizeof(double) * nobs, 256);
    const size_t extra = grid_extra(M, p, nstate) - (analysis_keepV(M, nstate, false) ? 0 : sizeof(double) * (size_t)M * M);
    const Plan pl = make_plan(M, batch, extra, wsb - ybytes);
    size_t off[7], total = 0;
    const size_t sizes[7] = {sizeof(double) * nobs * M, sizeof(double) * nobs, obs_mask ? (size_t)batch : 0,
                             sX * batch, wbar ? sw * batch : 0, sizeof(int) * (size_t)batch, wsb};
    for (int k = 0; k < 7; ++k) { off[k] = total; total += align_up(sizes[k] ? sizes[k] : 16, 256); }
    if ((rc = g_hpipe.reserve(total))) return rc;
    char* base = g_hpipe.arena;
    double* dYf = reinterpret_cast<double*>(base + off[0]);
    double* dyo = reinterpret_cast<double*>(base + off[1]);
    unsigned char* dmask = obs_mask ? reinterpret_cast<unsigned char*>(base + off[2]) : nullptr;
    double* dX = reinterpret_cast<double*>(base + off[3]);
    double* dwb = wbar ? reinterpret_cast<double*>(base + off[4]) : nullptr;
    int* dinfo = reinterpret_cast<int*>(base + off[5]);
    void* dwork = base + off[6];
    cudaStream_t sH = g_hpipe.s[0], sD = g_hpipe.s[1], sC = g_hpipe.sC;
    if ((rc = g_hpipe.events(2 * (size_t)pl.nsub + 1))) return rc;
    const cudaEvent_t* evH = g_hpipe.ev.data();
    const cudaEvent_t* evC = g_hpipe.ev.data() + pl.nsub;
    cudaEvent_t evF = g_hpipe.ev[2 * (size_t)pl.nsub];
    auto enqueue = [&]() -> int {
        CUDA_TRY(cudaMemcpyAsync(dYf, Yf, sizes[0], cudaMemcpyHostToDevice, sH));
        CUDA_TRY(cudaMemcpyAsync(dyo, yo, sizes[1], cudaMemcpyHostToDevice, sH));
        if (obs_mask) CUDA_TRY(cudaMemcpyAsync(dmask, obs_mask, sizes[2], cudaMemcpyHostToDevice, sH));
        CUDA_TRY(cudaEventRecord(evF, sH));
        for (int k = 0, c0 = 0; c0 < batch; ++k, c0 += pl.per) {
            const int nk = (batch - c0 < pl.per) ? batch - c0 : pl.per;
            CUDA_TRY(cudaMemcpyAsync(dX + (size_t)c0 * nstate * M, Xb + (size_t)c0 * nstate * M, sX * nk, cudaMemcpyHostToDevice, sH));
            CUDA_TRY(cudaEventRecord(evH[k], sH));
        }
        CUDA_TRY(cudaStreamWaitEvent(sC, evF, 0));                   // the fields before anything is gathered
        CUDA_TRY(cudaMemsetAsync(dinfo, 0, sizeof(int) * (size_t)batch, sC));
        HostCtx ctx{pl.per, 0, {}, {}, {}, sD, evH, evC};
        ctx.add(Xa, dX, sX);
        if (wbar) ctx.add(wbar, dwb, sw);
        if (info) ctx.add(info, dinfo, sizeof(int));
        PassHooks hooks{host_pre, host_post, &ctx};
        HooksGuard guard(&hooks);
        return letkf_analysis_grid(dYf, dyo, dmask, dX, M, V, Ny, Nx, nstate, hw, loc_kind, loc_scale, sigma_o, rho,
                                   dX, dwb, dinfo, dwork, wsb, sC);
    };
    rc = enqueue();
    const int launches = g_launches;
    const int dr = g_hpipe.drain();
    if (rc == 0) rc = dr;
    cudaError_t ce = cudaGetLastError();
    if (rc == 0 && ce != cudaSuccess) rc = (int)ce;
    g_launches = launches;
    return rc;
}

int letkf_probe_dfma(double* sink, int blocks, int threads, int iters,
                     unsigned long long* fma_count, void* stream)
{
    if (!sink) return -1;
    if (blocks < 1) return -2;
    if (threads < 1 || threads > 1024) return -3;
    if (iters < 0) return -4;
    probe_dfma_kernel<<<blocks, threads, 0, reinterpret_cast<cudaStream_t>(stream)>>>(sink, iters);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return (int)e;
    if (fma_count) *fma_count = (unsigned long long)blocks * threads * (unsigned long long)iters * 64ull;
    return LETKF_OK;
}

int letkf_last_launch_count(void) { return g_launches; }

int letkf_set_option(const char* name, int value)
{
    if (!name) return -1;
    std::lock_guard<std::mutex> lk(g_options_mu);
    Options& o = g_options;
    if (strcmp(name, "force_generic") == 0) { o.force_generic = value != 0; return LETKF_OK; }
    if (strcmp(name, "pipeline") == 0) { o.pipeline = value != 0; return LETKF_OK; }
    if (strcmp(name, "sub_chunk") == 0) { o.sub_chunk = value >= 1 ? value : 0; return LETKF_OK; }
    if (strcmp(name, "slots") == 0) { o.slots = value >= 2 ? value : 0; return LETKF_OK; }
    if (strcmp(name, "log_slots") == 0) { o.log_slots = value >= 2 ? value : 0; return LETKF_OK; }
    if (strcmp(name, "mid_reg") == 0) { o.mid_reg = (value >= 0 && value <= 2) ? value : 1; return LETKF_OK; }
    if (strcmp(name, "log_shrink") == 0) { o.log_shrink = value >= 1 ? value : 1; return LETKF_OK; }
    if (strcmp(name, "ql_tpb") == 0) { o.ql_tpb = (value == 32 || value == 64 || value == 96 || value == 128 || value == 192) ? value : 0; return LETKF_OK; }
    if (strcmp(name, "two_pass") == 0) { o.two_pass = (value == 0 || value == 1) ? value : -1; return LETKF_OK; }
    if (strcmp(name, "host_pass") == 0) { o.host_pass = value >= 1 ? value : 0; return LETKF_OK; }
    if (strcmp(name, "qform") == 0) { o.qform = value != 0; return LETKF_OK; }
    if (strcmp(name, "evec") == 0) { o.evec = value != 0; return LETKF_OK; }
    if (strcmp(name, "split") == 0) { o.split = value != 0; return LETKF_OK; }
    if (strcmp(name, "bigvec") == 0) { o.bigvec = value != 0; return LETKF_OK; }
    if (strcmp(name, "mid_split") == 0) { o.mid_split = value != 0; return LETKF_OK; }
    if (strcmp(name, "pack") == 0) { if (value < 0 || value > 3) return -2; o.pack = value; return LETKF_OK; }
    if (strcmp(name, "pair") == 0) { o.pair = (value == 0 || value == 1) ? value : -1; return LETKF_OK; }
    if (strcmp(name, "bisect") == 0) { o.bisect = (value == 0 || value == 1) ? value : -1; return LETKF_OK; }
    return -1;
}

int letkf_profile_enable(int on)
{
    const int prev = g_prof.on ? 1 : 0;
    g_prof.on = on != 0;
    g_prof.keep_pipeline = on == 2;
    return prev;
}

int letkf_profile_count(void) { return (int)g_prof.recs.size(); }

int letkf_profile_record(int idx, const char** name, float* ms)
{
    if (idx < 0 || idx >= (int)g_prof.recs.size()) return -1;
    const ProfRec& r = g_prof.recs[idx];
    cudaError_t e = cudaEventSynchronize(r.e1);
    if (e != cudaSuccess) return (int)e;
    float t = 0.f;
    e = cudaEventElapsedTime(&t, r.e0, r.e1);
    if (e != cudaSuccess) return (int)e;
    if (name) *name = r.name;
    if (ms) *ms = t;
    return LETKF_OK;
}

int letkf_profile_record_start(int idx, float* ms_from_first)
{
    if (idx < 0 || idx >= (int)g_prof.recs.size() || !ms_from_first) return -1;
    cudaError_t e = cudaEventSynchronize(g_prof.recs[idx].e0);
    if (e != cudaSuccess) return (int)e;
    e = cudaEventElapsedTime(ms_from_first, g_prof.recs[0].e0, g_prof.recs[idx].e0);
    return e == cudaSuccess ? LETKF_OK : (int)e;
}

long long letkf_profile_rotations(void)
{
    if (!g_prof.d_rot) return -1;
    unsigned long long v = 0;
    if (cudaMemcpy(&v, g_prof.d_rot, sizeof(v), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    return (long long)v;
}

long long letkf_profile_direct(void)
{
    if (!g_prof.d_rot) return -1;
    unsigned long long v = 0;
    if (cudaMemcpy(&v, g_prof.d_rot + 1, sizeof(v), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    return (long long)v;
}

const char* letkf_status_string(int status)
{
    static thread_local char buf[96];
    if (status == 0) return "ok";
    if (status == LETKF_ERR_STATIC_CAPACITY)
        return "batch too large for the static scratch array of letkf_syev_batched_static (letkf_syev_static_max_batch)";
    if (status < 0) {
        snprintf(buf, sizeof(buf), "invalid argument %d (1-based position in the call)", -status);
        return buf;
    }
    return cudaGetErrorString((cudaError_t)status);
}

int letkf_version(void) { return LETKF_VERSION; }

}  // extern "C"

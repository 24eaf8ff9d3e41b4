// letkf_api.cu -- the C ABI of libletkf (include/letkf.h): argument checking, workspace carving,
// dispatch on M, kernel launches.  No torch types; plain device pointers and sizes.
#include "../../include/letkf.h"

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <vector>

#include "common.cuh"
#include "ql_kernel.cuh"
#include "generic_kernels.cuh"
#include "fast_kernels.cuh"
#include "mid_kernels.cuh"

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
        if (!g_prof.d_rot) cudaMalloc(&g_prof.d_rot, sizeof(unsigned long long));
        cudaMemsetAsync(g_prof.d_rot, 0, sizeof(unsigned long long), st);
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

// bytes of workspace one matrix needs on the syev path
static size_t syev_bytes_per_matrix(int M)
{
    size_t s = 0;
    s += 2 * sizeof(double) * (size_t)M;                 // dws, ews
    s += sizeof(int) * (size_t)M;                        // perm
    s += 2 * sizeof(int);                                // nsweeps, flags
    s += sizeof(uint32_t) * (size_t)sweep_capacity(M);   // hdr
    s += sizeof(double2) * (size_t)log_capacity(M);      // rot
    return s;
}

// matrices processed per pass.  The workspace (dominated by the rotation log, 16*log_capacity(M)
// bytes per matrix) is sized for the whole batch up to WORK_CAP: ql_log_kernel costs the serial
// latency of one matrix's QL iteration whatever the batch (profiles/r01a), so passes are kept as
// few as the 180 GB of HBM allow.
static const size_t WORK_CAP = (size_t)8 << 30;
static int syev_chunk(int M, int batch)
{
    const size_t per = syev_bytes_per_matrix(M);
    size_t c = WORK_CAP / per;
    if (c < 1024) c = 1024;
    if (c > (size_t)batch) c = (size_t)batch;
    if (c < 1) c = 1;
    return (int)c;
}

static int g_log_shrink = 1;             // letkf_set_option("log_shrink", k): tests force the slow path

static size_t carve(Workspace& ws, void* base, int M, int chunk)
{
    char* p = reinterpret_cast<char*>(base);
    size_t off = 0;
    auto take = [&](size_t bytes) { char* q = p ? p + off : nullptr; off = align_up(off + bytes, 256); return q; };
    ws.swcap = sweep_capacity(M);
    ws.logcap = log_capacity(M) / g_log_shrink;       // (the memory is still sized for the full log)
    ws.rot_counter = g_prof.on ? g_prof.d_rot : nullptr;
    ws.dws     = reinterpret_cast<double*>(take(sizeof(double) * (size_t)M * chunk));
    ws.ews     = reinterpret_cast<double*>(take(sizeof(double) * (size_t)M * chunk));
    ws.perm    = reinterpret_cast<int*>(take(sizeof(int) * (size_t)M * chunk));
    ws.nsweeps = reinterpret_cast<int*>(take(sizeof(int) * (size_t)chunk));
    ws.flags   = reinterpret_cast<int*>(take(sizeof(int) * (size_t)chunk));
    ws.hdr     = reinterpret_cast<uint32_t*>(take(sizeof(uint32_t) * (size_t)ws.swcap * chunk));
    ws.rot     = reinterpret_cast<double2*>(take(sizeof(double2) * (size_t)ws.logcap * chunk));
    return off;
}

// the records of matrices b0 ... of a carved workspace
static Workspace ws_slice(const Workspace& w, int M, int b0)
{
    Workspace s = w;
    s.dws += (size_t)b0 * M;
    s.ews += (size_t)b0 * M;
    s.perm += (size_t)b0 * M;
    s.nsweeps += b0;
    s.flags += b0;
    s.hdr += (size_t)b0 * w.swcap;
    s.rot += (size_t)b0 * w.logcap;
    return s;
}

static inline bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

#define LAUNCH_CHECK()                                         \
    do {                                                       \
        cudaError_t e_ = cudaGetLastError();                   \
        if (e_ != cudaSuccess) return (int)e_;                 \
        ++g_launches;                                          \
    } while (0)

template <typename K>
static cudaError_t allow_smem(K kernel, size_t bytes)
{
    cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (bytes <= 48 * 1024) return cudaSuccess;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

static int g_mid_reg = 1;                // letkf_set_option("mid_reg", 0 / 1 / 2): 64 < M <= 160 reduced in shared memory / registers up to M = 128 / registers
static bool g_force_generic = false;     // letkf_set_option("force_generic", 1): tests only

// a1/a2 inputs when the matrix is to be formed from the LETKF observations instead of read
struct GramArgs { const double* Yb; const double* d; const double* r; int p; double shift; double* gout; GridArgs grid; };

static int g_split = 0;                  // letkf_set_option("split", 1): three-kernel tridiagonalisation for M in (48, 64] (slower so far)

template <int MT>
static int fast_tridiag_run(const double* A, double* V, Workspace ws, int M, int n, cudaStream_t st,
                            const GramArgs* gram)
{
    const size_t smem = fast_tridiag_smem<MT>();
    cudaError_t ce;
    if constexpr (MT == 64) {
        if (g_split && M > 34 && sizeof(double2) * (size_t)ws.logcap >= sizeof(double) * SPLIT_DOUBLES) {
            if (gram) {
                if ((ce = allow_smem(fast_tridiag_formq<MT, true, true>, smem)) != cudaSuccess) return (int)ce;
                KLAUNCH("fast_tridiag_head<gram>", st,
                        fast_tridiag_formq<MT, true, true><<<n, FastCfg<MT>::NT, smem, st>>>(
                            nullptr, V, ws, M, gram->Yb, gram->d, gram->r, gram->p, gram->shift, gram->gout, gram->grid));
            } else {
                if ((ce = allow_smem(fast_tridiag_formq<MT, false, true>, smem)) != cudaSuccess) return (int)ce;
                KLAUNCH("fast_tridiag_head", st,
                        fast_tridiag_formq<MT, false, true><<<n, FastCfg<MT>::NT, smem, st>>>(
                            A, V, ws, M, nullptr, nullptr, nullptr, 0, 0.0, nullptr, GridArgs{}));
            }
            KLAUNCH("fast_tridiag_tail", st, fast_tridiag_tail<<<n, 32, sizeof(double) * (640 + 176), st>>>(ws, M));
            const size_t qs = sizeof(double) * (2304 + 64);
            if ((ce = allow_smem(fast_formq, qs)) != cudaSuccess) return (int)ce;
            KLAUNCH("fast_formq", st, fast_formq<<<2 * n, 32, qs, st>>>(V, ws, M));
            return 0;
        }
    }
    if (gram) {
        if ((ce = allow_smem(fast_tridiag_formq<MT, true>, smem)) != cudaSuccess) return (int)ce;
        KLAUNCH("fast_tridiag_formq<gram>", st,
                fast_tridiag_formq<MT, true><<<n, FastCfg<MT>::NT, smem, st>>>(
                    nullptr, V, ws, M, gram->Yb, gram->d, gram->r, gram->p, gram->shift, gram->gout, gram->grid));
    } else {
        if ((ce = allow_smem(fast_tridiag_formq<MT, false>, smem)) != cudaSuccess) return (int)ce;
        KLAUNCH("fast_tridiag_formq", st,
                fast_tridiag_formq<MT, false><<<n, FastCfg<MT>::NT, smem, st>>>(
                    A, V, ws, M, nullptr, nullptr, nullptr, 0, 0.0, nullptr, GridArgs{}));
    }
    return 0;
}

template <int MT>
static int fast_apply_run(double* V, Workspace ws, int M, int n, cudaStream_t st, const EpiArgs* ep)
{
    cudaError_t ce;
    if (ep) {
        const size_t smem = fast_apply_smem<MT>(ws.swcap) + fast_epi_smem<MT>(ep->ns);
        if ((ce = allow_smem(fast_apply<MT, true>, smem)) != cudaSuccess) return (int)ce;
        KLAUNCH("fast_apply<epilogue>", st, fast_apply<MT, true><<<n, FastCfg<MT>::NT, smem, st>>>(V, ws, M, *ep));
    } else {
        const size_t smem = fast_apply_smem<MT>(ws.swcap);
        if ((ce = allow_smem(fast_apply<MT, false>, smem)) != cudaSuccess) return (int)ce;
        KLAUNCH("fast_apply", st, fast_apply<MT, false><<<n, FastCfg<MT>::NT, smem, st>>>(V, ws, M, EpiArgs{}));
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// The EVD of n matrices as three stages.  stage_T: a3 (+ a1, a2 with `gram`) and the explicit Q;
// stage_QL: a4, the logged QL iteration; stage_AP: a5, replay of the log on Q, eigenvalue sort.
// ws is the workspace slice of these n matrices.
static int stage_T(const double* A, int M, int n, double* V, Workspace ws, cudaStream_t st,
                   const GramArgs* gram)
{
    if (fast_supported(M) && !g_force_generic) {
        switch (fast_bucket(M)) {
            case 16: return fast_tridiag_run<16>(A, V, ws, M, n, st, gram);
            case 32: return fast_tridiag_run<32>(A, V, ws, M, n, st, gram);
            case 48: return fast_tridiag_run<48>(A, V, ws, M, n, st, gram);
            default: return fast_tridiag_run<64>(A, V, ws, M, n, st, gram);
        }
    }
    if (gram) {
        KLAUNCH("generic_gram", st,
                generic_gram<<<n, 256, 0, st>>>(gram->Yb, gram->d, gram->r, M, gram->p, gram->shift, V, gram->gout));
        A = V;
    }
    if (mid_supported(M) && !g_force_generic) {          // matrix resident in shared memory
        cudaError_t ce;
        const size_t smem = mid_tridiag_smem(M);
        const int mt = mid_threads(M);
        // registers hold the matrix up to M = 128 (measured, batch 2^26/M^2: M = 96 6.58 -> 5.12 ms, M = 128 9.42 -> 7.57 ms);
        // at MT = 160 the 80 matrix registers of a thread spill under the 102 a CTA of 640 allows and
        // the shared-memory form is as fast (10.5 vs 10.9 ms): mid_reg = 1 (default) / 2 (force) / 0 (never)
        const bool reg = g_mid_reg == 2 || (g_mid_reg == 1 && mt <= 128);
        auto kern = reg ? (mt == 96 ? mid_tridiag_formq_reg<96> : (mt == 128 ? mid_tridiag_formq_reg<128> : mid_tridiag_formq_reg<160>))
                        : (mt == 96 ? mid_tridiag_formq<96> : (mt == 128 ? mid_tridiag_formq<128> : mid_tridiag_formq<160>));
        if ((ce = allow_smem(kern, smem)) != cudaSuccess) return (int)ce;
        KLAUNCH("mid_tridiag_formq", st, kern<<<n, MID_TPR * mt, smem, st>>>(A, V, ws, M));
        return 0;
    }
    const size_t td_smem = sizeof(double) * ((4 + GEN_QK) * (size_t)M + GEN_NT / 32);
    KLAUNCH("generic_tridiag_formq", st, generic_tridiag_formq<<<n, GEN_NT, td_smem, st>>>(A, V, ws, M));
    return 0;
}

static int g_ql_tpb = 0;                 // letkf_set_option("ql_tpb", 32/64/96): 0 = by size

template <int TPB>
static int ql_run(int M, int n, double* w, int* info, Workspace ws, cudaStream_t st)
{
    cudaError_t ce;
    const size_t ql_smem = sizeof(double) * 2 * (size_t)M * TPB;
    if ((ce = allow_smem(ql_log_kernel<TPB>, ql_smem)) != cudaSuccess) return (int)ce;
    const int qblocks = (n + TPB - 1) / TPB;
    KLAUNCH("ql_log_kernel", st, ql_log_kernel<TPB><<<qblocks, TPB, ql_smem, st>>>(ws, M, n, w, info));
    return 0;
}

static int stage_QL(int M, int n, double* w, int* info, Workspace ws, cudaStream_t st)
{
    int tpb = g_ql_tpb ? g_ql_tpb : (M <= 64 ? 64 : 32);
    while (tpb > 32 && sizeof(double) * 2 * (size_t)M * tpb > 200 * 1024) tpb -= 32;
    switch (tpb) {
        case 96: return ql_run<96>(M, n, w, info, ws, st);
        case 64: return ql_run<64>(M, n, w, info, ws, st);
        default: return ql_run<32>(M, n, w, info, ws, st);
    }
}

static int stage_AP(int M, int n, double* w, double* V, int* info, Workspace ws, cudaStream_t st,
                    const EpiArgs* ep = nullptr)
{
    const size_t ap_smem = sizeof(double) * (5 * (size_t)M + 2 * 32 * 33);
    if (fast_supported(M) && !g_force_generic) {
        int rc = 0;
        switch (fast_bucket(M)) {
            case 16: rc = fast_apply_run<16>(V, ws, M, n, st, ep); break;
            case 32: rc = fast_apply_run<32>(V, ws, M, n, st, ep); break;
            case 48: rc = fast_apply_run<48>(V, ws, M, n, st, ep); break;
            default: rc = fast_apply_run<64>(V, ws, M, n, st, ep); break;
        }
        if (rc) return rc;
        // finisher for matrices whose rotation log overflowed (normally none: exits at once)
        KLAUNCH("generic_apply(flagged)", st,
                generic_apply<<<(n < 296 ? n : 296), GEN_NT, ap_smem, st>>>(V, w, ws, M, n, info, /*only_flagged=*/1, /*q_rowmajor=*/1));
        return 0;
    }
    if (mid_supported(M) && !g_force_generic) {
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
        KLAUNCH("generic_apply(flagged)", st,
                generic_apply<<<(n < 296 ? n : 296), GEN_NT, ap_smem, st>>>(V, w, ws, M, n, info, /*only_flagged=*/1, /*q_rowmajor=*/0));
        return 0;
    }
    KLAUNCH("generic_apply", st, generic_apply<<<n, GEN_NT, ap_smem, st>>>(V, w, ws, M, n, info, 0, 0));
    return 0;
}

// ---------------------------------------------------------------------------------------------
// Private streams of the calling host thread.  A pass over n matrices is cut into sub-chunks that
// flow through three stages on separate streams: ql_log_kernel is bound by the serial latency of
// one matrix's iteration and keeps one warp per SM sub-partition busy at most, so it runs beside
// the ALU-bound stage_T / stage_AP kernels of the neighbouring sub-chunks (highest priority, so a
// ready QL block takes the first free slot).  stage_T outranks stage_AP: every QL kernel should
// start as early as possible, the apply kernels fill the machine behind them.  Everything is forked from and joined back into the
// caller's stream with events: the caller sees plain stream order.
struct Pipe {
    int dev = -1;
    cudaStream_t sT[2] = {nullptr, nullptr}, sA[4] = {};
    cudaStream_t sQ[16] = {};          // one per sub-chunk: all QL kernels of a pass run side by side
    std::vector<cudaEvent_t> ev;
    size_t used = 0;
    int init()
    {
        int d = 0;
        cudaError_t ce = cudaGetDevice(&d);
        if (ce != cudaSuccess) return (int)ce;
        if (d == dev) return 0;
        int least = 0, greatest = 0;
        cudaDeviceGetStreamPriorityRange(&least, &greatest);
        const int mid = (greatest < least) ? greatest + 1 : greatest;
        for (int k = 0; k < 2; ++k) {
            if ((ce = cudaStreamCreateWithPriority(&sT[k], cudaStreamNonBlocking, mid)) != cudaSuccess) return (int)ce;
        }
        for (int k = 0; k < 4; ++k)
            if ((ce = cudaStreamCreateWithPriority(&sA[k], cudaStreamNonBlocking, least)) != cudaSuccess) return (int)ce;
        for (int k = 0; k < 16; ++k)
            if ((ce = cudaStreamCreateWithPriority(&sQ[k], cudaStreamNonBlocking, greatest)) != cudaSuccess) return (int)ce;
        ev.clear();
        used = 0;
        dev = d;
        return 0;
    }
    cudaEvent_t event()
    {
        if (used == ev.size()) {
            cudaEvent_t e;
            cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
            ev.push_back(e);
        }
        return ev[used++];
    }
    // `to` waits for everything enqueued on `from` so far
    void link(cudaStream_t from, cudaStream_t to)
    {
        cudaEvent_t e = event();
        cudaEventRecord(e, from);
        cudaStreamWaitEvent(to, e, 0);
    }
};
static thread_local Pipe g_pipe;

static int g_pipeline = 1;               // letkf_set_option("pipeline", 0): one stream, one chunk
static const int PIPE_MIN_SUB = 1024;    // smallest sub-chunk worth a launch of its own
static const int PIPE_MAX_SUB = 16;      // = number of QL streams
static thread_local int g_max_sub = 8;   // sub-chunks per pass: 8 for device calls (measured best), 16 for the
                                         // host entry points (finer copy/compute overlap: shorter head and tail)

// One pass: n matrices whose workspace records are ws[0..n).  stageT(b0, nk, stream) enqueues the
// first stage of matrices [b0, b0+nk); post(b0, nk, stream) whatever follows stage_AP (the
// analysis epilogue) or nothing.
static EpiArgs epi_slice(const EpiArgs& e, int M, int b0)
{
    EpiArgs s = e;
    s.lam += (size_t)b0 * M;
    s.g += (size_t)b0 * M;
    s.Xb += (size_t)b0 * e.ns * M;
    s.Xa += (size_t)b0 * e.ns * M;
    if (s.wbar) s.wbar += (size_t)b0 * M;
    return s;
}

// Sub-chunks of a pass of n matrices: nsub pieces of `per` matrices (the last one shorter).
static void pass_partition(int n, int& nsub, int& per)
{
    nsub = (g_pipeline && (!g_prof.on || g_prof.keep_pipeline)) ? n / PIPE_MIN_SUB : 1;
    if (nsub > g_max_sub) nsub = g_max_sub;
    if (nsub < 1) nsub = 1;
    per = (n + nsub - 1) / nsub;
}

// ep0: a6-a9 fused into the apply kernel (pointers of matrix 0 of the pass), or NULL.
template <class FT, class FP>
static int run_pass(int M, int n, double* w, double* V, int* info, const Workspace& ws,
                    cudaStream_t st, FT stageT, FP post, const EpiArgs* ep0 = nullptr)
{
    int nsub, per;
    pass_partition(n, nsub, per);
    if (nsub < 2) {
        int rc = stageT(0, n, st);
        if (rc) return rc;
        if ((rc = stage_QL(M, n, w, info, ws, st))) return rc;
        if ((rc = stage_AP(M, n, w, V, info, ws, st, ep0))) return rc;
        return post(0, n, st);
    }
    Pipe& P = g_pipe;
    int rc = P.init();
    if (rc) return rc;
    P.used = 0;
    for (int k = 0; k < 2; ++k) P.link(st, P.sT[k]);
    for (int k = 0; k < 4; ++k) P.link(st, P.sA[k]);
    for (int k = 0; k < nsub; ++k) P.link(st, P.sQ[k]);
    for (int k = 0, b0 = 0; b0 < n; ++k, b0 += per) {
        const int nk = (n - b0 < per) ? n - b0 : per;
        const int s = k & 1;
        const Workspace wk = ws_slice(ws, M, b0);
        int* infok = info ? info + b0 : nullptr;
        if ((rc = stageT(b0, nk, P.sT[s]))) return rc;
        P.link(P.sT[s], P.sQ[k]);
        if ((rc = stage_QL(M, nk, w + (size_t)b0 * M, infok, wk, P.sQ[k]))) return rc;
        cudaStream_t sa = P.sA[k & 3];
        P.link(P.sQ[k], sa);
        EpiArgs epk;
        if (ep0) epk = epi_slice(*ep0, M, b0);
        if ((rc = stage_AP(M, nk, w + (size_t)b0 * M, V + (size_t)b0 * M * M, infok, wk, sa, ep0 ? &epk : nullptr))) return rc;
        if ((rc = post(b0, nk, sa))) return rc;
    }
    for (int k = 0; k < 2; ++k) P.link(P.sT[k], st);
    for (int k = 0; k < 4; ++k) P.link(P.sA[k], st);
    for (int k = 0; k < nsub; ++k) P.link(P.sQ[k], st);
    return 0;
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

}  // namespace letkf

using namespace letkf;

extern "C" {

size_t letkf_syev_workspace_bytes(int M, int batch)
{
    if (M < 1 || M > LETKF_MAX_M || batch < 1) return 0;
    Workspace ws;
    return carve(ws, nullptr, M, syev_chunk(M, batch));
}

// Hooks of the host-buffer entry points: pre(b0, nk, s) is enqueued on the stream of a sub-chunk's
// first kernel before it (wait for the sub-chunk's inputs), post(b0, nk, s) after its last kernel
// (start the read-back).  b0 counts from the start of the pass.
struct PassHooks {
    int (*pre)(void* ctx, int b0, int nk, cudaStream_t s);
    int (*post)(void* ctx, int b0, int nk, cudaStream_t s);
    void* ctx;
};

static thread_local const PassHooks* g_analysis_hooks = nullptr;   // set by the host entry point only

// one pass (n <= syev_chunk matrices, workspace carved for them) of the EVD on device buffers
static int syev_pass(const double* A, int M, int n, double* w, double* V, int* info, const Workspace& ws,
                     cudaStream_t st, const PassHooks* hooks)
{
    auto stageT = [&](int c0, int nk, cudaStream_t s) {
        if (hooks) { const int rc = hooks->pre(hooks->ctx, c0, nk, s); if (rc) return rc; }
        return stage_T(A + (size_t)c0 * M * M, M, nk, V + (size_t)c0 * M * M, ws_slice(ws, M, c0), s, nullptr);
    };
    auto post = [&](int c0, int nk, cudaStream_t s) { return hooks ? hooks->post(hooks->ctx, c0, nk, s) : 0; };
    return run_pass(M, n, w, V, info, ws, st, stageT, post);
}

int letkf_syev_batched(const double* A, int M, int batch, double* w, double* V, int* info,
                       void* work, size_t work_bytes, void* stream)
{
    g_launches = 0;
    if (M < 1 || M > LETKF_MAX_M) return -2;
    if (batch < 0) return -3;
    if (batch == 0) return LETKF_OK;
    if (!A || misaligned(A)) return -1;
    if (!w || misaligned(w)) return -4;
    if (!V || misaligned(V)) return -5;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    prof_reset(st);

    const int chunk = syev_chunk(M, batch);
    Workspace ws;
    const size_t need = carve(ws, nullptr, M, chunk);
    ScopedWork sw;
    int rc = sw.acquire(work, work_bytes, need, st, 7);
    if (rc) return rc;
    carve(ws, sw.ptr, M, chunk);

    for (int b0 = 0; b0 < batch; b0 += chunk) {
        const int n = (batch - b0 < chunk) ? batch - b0 : chunk;
        rc = syev_pass(A + (size_t)b0 * M * M, M, n, w + (size_t)b0 * M, V + (size_t)b0 * M * M,
                       info ? info + b0 : nullptr, ws, st, nullptr);
        if (rc) return rc;
    }
    return LETKF_OK;
}

size_t letkf_analysis_workspace_bytes(int M, int p, int nstate, int batch)
{
    (void)p; (void)nstate;
    if (M < 1 || M > LETKF_MAX_M || batch < 1) return 0;
    const int chunk = syev_chunk(M, batch);
    Workspace ws;
    size_t s = carve(ws, nullptr, M, chunk);
    s += align_up(sizeof(double) * (size_t)M * M * chunk, 256);   // Q / V
    s += align_up(sizeof(double) * (size_t)M * chunk, 256);       // lam
    s += align_up(sizeof(double) * (size_t)M * chunk, 256);       // g
    return s;
}

// does the grid form run with the gather fused into the tridiagonalisation kernel?
static bool grid_fused(int M, int nstate) { return fast_supported(M) && !g_force_generic && nstate <= EPI_NS_MAX; }

size_t letkf_analysis_grid_workspace_bytes(int M, int V, int Ny, int Nx, int hw, int nstate)
{
    if (M < 2 || M > LETKF_MAX_M || V < 1 || Ny < 1 || Nx < 1 || hw < 0 || nstate < 1) return 0;
    const long npts = (long)Ny * Nx;
    if (npts > 0x7fffffffL) return 0;
    const int batch = (int)npts, p = V * (2 * hw + 1) * (2 * hw + 1);
    size_t s = align_up(letkf_analysis_workspace_bytes(M, p, nstate, batch), 256);
    s += align_up(sizeof(double) * (size_t)V * npts, 256);                                   // ybar
    const int chunk = syev_chunk(M, batch);                                                  // materialised Y_loc
    s += align_up(sizeof(double) * (size_t)p * M * chunk, 256) + 2 * align_up(sizeof(double) * (size_t)p * chunk, 256);
    return s;
}

// a1-a9 for `batch` grid points.  Either (Yb, d, rinv_loc) or `grid` (then gYb/gd/gr are scratch
// for the materialised local observations of one pass, used when the gather cannot be fused).
static int analysis_core(const double* Yb, const double* d, const double* rinv_loc, const GridArgs* grid,
                         double* gYb, double* gd, double* gr,
                         const double* Xb, int M, int p, int nstate, int batch, double rho,
                         double* Xa, double* W, double* wbar, int* info,
                         void* work, size_t work_bytes, int work_argpos, cudaStream_t st)
{
    const int chunk = syev_chunk(M, batch);
    const size_t need = letkf_analysis_workspace_bytes(M, p, nstate, batch);
    ScopedWork sw;
    int rc = sw.acquire(work, work_bytes, need, st, work_argpos);
    if (rc) return rc;
    Workspace ws;
    size_t off = carve(ws, sw.ptr, M, chunk);
    char* base = reinterpret_cast<char*>(sw.ptr);
    double* Vbuf = reinterpret_cast<double*>(base + off); off += align_up(sizeof(double) * (size_t)M * M * chunk, 256);
    double* lam  = reinterpret_cast<double*>(base + off); off += align_up(sizeof(double) * (size_t)M * chunk, 256);
    double* gbuf = reinterpret_cast<double*>(base + off);

    const double shift = (double)(M - 1) / rho;
    cudaError_t ce;
    const size_t ep_smem = sizeof(double) * (2 * (size_t)M + 2 * (size_t)nstate + 2 * (size_t)nstate * M);
    if (ep_smem > 200 * 1024) return -7;
    if ((ce = allow_smem(generic_epilogue, ep_smem)) != cudaSuccess) return (int)ce;
    const bool fuse_gather = grid && !W && grid_fused(M, nstate);

    for (int b0 = 0; b0 < batch; b0 += chunk) {
        const int n = (batch - b0 < chunk) ? batch - b0 : chunk;
        // local observations of this pass: the caller's arrays, or the scratch the gather fills
        const double* Ybc = grid ? gYb : Yb + (size_t)b0 * p * M;
        const double* dc = grid ? gd : d + (size_t)b0 * p;
        const double* rc_ = grid ? gr : rinv_loc + (size_t)b0 * p;
        const double* Xbc = Xb + (size_t)b0 * nstate * M;
        double* Xac = Xa + (size_t)b0 * nstate * M;
        double* Wc = W ? W + (size_t)b0 * M * M : nullptr;
        double* wbc = wbar ? wbar + (size_t)b0 * M : nullptr;
        int* infoc = info ? info + b0 : nullptr;

        auto stageT = [&](int c0, int nk, cudaStream_t s) {
            if (g_analysis_hooks) {
                const int hrc = g_analysis_hooks->pre(g_analysis_hooks->ctx, b0 + c0, nk, s);
                if (hrc) return hrc;
            }
            GramArgs ga{Ybc + (size_t)c0 * p * M, dc + (size_t)c0 * p, rc_ + (size_t)c0 * p, p, shift,
                        gbuf + (size_t)c0 * M, GridArgs{}};
            if (grid) {
                GridArgs gk = *grid;
                gk.point0 = grid->point0 + b0 + c0;
                if (fuse_gather) {
                    ga.grid = gk;
                } else {
                    KLAUNCH("grid_gather", s,
                            grid_gather<<<nk, 256, 0, s>>>(gk, M, p, gYb + (size_t)c0 * p * M, gd + (size_t)c0 * p,
                                                           gr + (size_t)c0 * p));
                }
            }
            double* Vk = Vbuf + (size_t)c0 * M * M;
            return stage_T(Vk, M, nk, Vk, ws_slice(ws, M, c0), s, &ga);
        };
        // a6-a9: fused into fast_apply when W is not wanted (V then never leaves the SM); the
        // any-M kernel otherwise, and for the grid points the slow path finished.
        const bool fused = !Wc && fast_supported(M) && !g_force_generic && nstate <= EPI_NS_MAX;
        auto post = [&](int c0, int nk, cudaStream_t s) -> int {
            const int gridsz = fused ? (nk < 296 ? nk : 296) : nk;
            KLAUNCH(fused ? "generic_epilogue(flagged)" : "generic_epilogue", s,
                    generic_epilogue<<<gridsz, 256, ep_smem, s>>>(
                        Vbuf + (size_t)c0 * M * M, lam + (size_t)c0 * M, gbuf + (size_t)c0 * M,
                        Xbc + (size_t)c0 * nstate * M, M, nstate, nk, Xac + (size_t)c0 * nstate * M,
                        Wc ? Wc + (size_t)c0 * M * M : nullptr, wbc ? wbc + (size_t)c0 * M : nullptr,
                        fused ? ws.flags + c0 : nullptr));
            return g_analysis_hooks ? g_analysis_hooks->post(g_analysis_hooks->ctx, b0 + c0, nk, s) : 0;
        };
        EpiArgs ep{lam, gbuf, Xbc, Xac, wbc, nstate};
        rc = run_pass(M, n, lam, Vbuf, infoc, ws, st, stageT, post, fused ? &ep : nullptr);
        if (rc) return rc;
    }
    return LETKF_OK;
}

int letkf_analysis_batched(const double* Yb, const double* d, const double* rinv_loc,
                           const double* Xb, int M, int p, int nstate, int batch, double rho,
                           double* Xa, double* W, double* wbar, int* info,
                           void* work, size_t work_bytes, void* stream)
{
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
    return analysis_core(Yb, d, rinv_loc, nullptr, nullptr, nullptr, nullptr, Xb, M, p, nstate, batch, rho,
                         Xa, W, wbar, info, work, work_bytes, 14, st);
}

int letkf_analysis_grid(const double* Yf, const double* yo, const unsigned char* obs_mask, const double* Xb,
                        int M, int V, int Ny, int Nx, int nstate, int hw, int loc_kind, double loc_scale,
                        double sigma_o, double rho, double* Xa, double* wbar, int* info,
                        void* work, size_t work_bytes, void* stream)
{
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
    const size_t need = letkf_analysis_grid_workspace_bytes(M, V, Ny, Nx, hw, nstate);
    ScopedWork sw;
    int rc = sw.acquire(work, work_bytes, need, st, 18);
    if (rc) return rc;
    // carve: [analysis workspace][ybar][materialised Y_loc of one pass]
    const size_t wa = align_up(letkf_analysis_workspace_bytes(M, p, nstate, batch), 256);
    char* base = reinterpret_cast<char*>(sw.ptr);
    double* ybar = reinterpret_cast<double*>(base + wa);
    size_t off = wa + align_up(sizeof(double) * (size_t)V * batch, 256);
    const int chunk = syev_chunk(M, batch);
    double* gYb = reinterpret_cast<double*>(base + off); off += align_up(sizeof(double) * (size_t)p * M * chunk, 256);
    double* gd = reinterpret_cast<double*>(base + off);  off += align_up(sizeof(double) * (size_t)p * chunk, 256);
    double* gr = reinterpret_cast<double*>(base + off);
    const long nobs = (long)V * batch;
    KLAUNCH("grid_obs_mean", st, grid_obs_mean<<<(unsigned)((nobs + 7) / 8), 256, 0, st>>>(Yf, ybar, nobs, M));
    GridArgs g{Yf, ybar, yo, obs_mask, V, Ny, Nx, hw, loc_kind, loc_scale, 1.0 / (sigma_o * sigma_o), 0};
    rc = analysis_core(nullptr, nullptr, nullptr, &g, gYb, gd, gr, Xb, M, p, nstate, batch, rho,
                       Xa, nullptr, wbar, info, base, wa, 18, st);
    return rc;
}

// ---- host-buffer entry points -----------------------------------------------------------------
// A pass of the batch lives on the device at a time; the sub-chunks of the kernel pipeline are
// copied in one after the other on a copy-in stream, each sub-chunk's first kernel waits for its
// own copy only, and its read-back starts on a copy-out stream as soon as its last kernel is done:
// both copy engines and the SMs overlap (PCIe is full duplex).  The device staging arena is kept by the calling host thread between calls
// (letkf_host_release() frees it); the call returns after the last byte has reached the host.
struct HostPipe {
    int dev = -1;
    cudaStream_t s[2] = {nullptr, nullptr};
    cudaStream_t sC = nullptr;    // the stream the kernels of a host call are forked from
    std::vector<cudaEvent_t> ev;
    void events(size_t n)
    {
        while (ev.size() < n) {
            cudaEvent_t e;
            cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
            ev.push_back(e);
        }
    }
    char* arena = nullptr;        // device staging memory, grown on demand and kept between calls
    size_t arena_bytes = 0;       // (re-allocating > 1 GB per call costs more than the whole EVD)
    int reserve(size_t bytes)
    {
        if (bytes <= arena_bytes) return 0;
        if (arena) cudaFree(arena);
        arena = nullptr;
        arena_bytes = 0;
        cudaError_t ce = cudaMalloc(reinterpret_cast<void**>(&arena), bytes);
        if (ce != cudaSuccess) return (int)ce;
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
        arena = nullptr;            // memory of another device is left to that device's context
        arena_bytes = 0;
        for (int k = 0; k < 2; ++k)
            if ((ce = cudaStreamCreateWithFlags(&s[k], cudaStreamNonBlocking)) != cudaSuccess) return (int)ce;
        if ((ce = cudaStreamCreateWithFlags(&sC, cudaStreamNonBlocking)) != cudaSuccess) return (int)ce;
        ev.clear();
        dev = d;
        return 0;
    }
};
static thread_local HostPipe g_hpipe;

// the host entry points cut a pass into up to PIPE_MAX_SUB sub-chunks for the duration of the call
struct HostSubChunks {
    int old;
    HostSubChunks() : old(g_max_sub) { g_max_sub = PIPE_MAX_SUB; }
    ~HostSubChunks() { g_max_sub = old; }
};

// context of the copy hooks of letkf_syev_batched_host
struct SyevHostCtx {
    int M, per;                       // sub-chunk size of the pass
    const double* hA; double* hw; double* hV; int* hinfo;      // host, at the start of the pass
    double* dV; double* dw; int* dinfo;                          // device, at the start of the pass
    cudaStream_t sD;                  // read-back stream
    std::vector<cudaEvent_t>* evH;    // evH[k]: inputs of sub-chunk k are on the device
    std::vector<cudaEvent_t>* evC;    // evC[k]: outputs of sub-chunk k are final
};
static int syev_host_pre(void* c, int b0, int, cudaStream_t s)
{
    SyevHostCtx* x = static_cast<SyevHostCtx*>(c);
    return (int)cudaStreamWaitEvent(s, (*x->evH)[b0 / x->per], 0);
}
static int syev_host_post(void* c, int b0, int nk, cudaStream_t s)
{
    SyevHostCtx* x = static_cast<SyevHostCtx*>(c);
    const int M = x->M;
    cudaEvent_t e = (*x->evC)[b0 / x->per];
    cudaError_t ce;
    if ((ce = cudaEventRecord(e, s)) != cudaSuccess) return (int)ce;
    if ((ce = cudaStreamWaitEvent(x->sD, e, 0)) != cudaSuccess) return (int)ce;
    if ((ce = cudaMemcpyAsync(x->hV + (size_t)b0 * M * M, x->dV + (size_t)b0 * M * M,
                              sizeof(double) * (size_t)nk * M * M, cudaMemcpyDeviceToHost, x->sD)) != cudaSuccess) return (int)ce;
    if ((ce = cudaMemcpyAsync(x->hw + (size_t)b0 * M, x->dw + (size_t)b0 * M,
                              sizeof(double) * (size_t)nk * M, cudaMemcpyDeviceToHost, x->sD)) != cudaSuccess) return (int)ce;
    if (x->hinfo &&
        (ce = cudaMemcpyAsync(x->hinfo + b0, x->dinfo + b0, sizeof(int) * (size_t)nk, cudaMemcpyDeviceToHost, x->sD)) != cudaSuccess)
        return (int)ce;
    return 0;
}

int letkf_syev_batched_host(const double* A, int M, int batch, double* w, double* V, int* info)
{
    g_launches = 0;
    if (M < 1 || M > LETKF_MAX_M) return -2;
    if (batch < 0) return -3;
    if (batch == 0) return LETKF_OK;
    if (!A) return -1;
    if (!w) return -4;
    if (!V) return -5;
    int rc = g_hpipe.init();
    if (rc) return rc;
    // One pass of up to syev_chunk matrices lives on the device at a time.  Its sub-chunks (the
    // ones the kernel pipeline uses) are copied in one after the other on the copy-in stream; each
    // sub-chunk's first kernel waits for its own copy only, and its read-back starts on the
    // copy-out stream as soon as its last kernel is done: both copy engines and the SMs overlap.
    const int chunk = syev_chunk(M, batch);
    const size_t mat = sizeof(double) * (size_t)M * M, vec = sizeof(double) * (size_t)M;
    Workspace ws;
    const size_t wsb = align_up(carve(ws, nullptr, M, chunk), 256);
    const size_t oV = 0, ow = align_up(mat * chunk, 256), oi = ow + align_up(vec * chunk, 256);
    const size_t owk = oi + align_up(sizeof(int) * (size_t)chunk, 256);
    if ((rc = g_hpipe.reserve(owk + wsb))) return rc;
    char* base = g_hpipe.arena;
    double* dV = reinterpret_cast<double*>(base + oV);
    double* dw = reinterpret_cast<double*>(base + ow);
    int* dinfo = reinterpret_cast<int*>(base + oi);
    carve(ws, base + owk, M, chunk);
    cudaStream_t sH = g_hpipe.s[0], sD = g_hpipe.s[1], sC = g_hpipe.sC;
    int launches = 0;
    HostSubChunks max_sub_guard;
    for (int b0 = 0; b0 < batch && rc == 0; b0 += chunk) {
        const int n = (batch - b0 < chunk) ? batch - b0 : chunk;
        int nsub, per;
        prof_reset(sC);
        pass_partition(n, nsub, per);
        g_hpipe.events(2 * nsub);
        std::vector<cudaEvent_t> evH(g_hpipe.ev.begin(), g_hpipe.ev.begin() + nsub);
        std::vector<cudaEvent_t> evC(g_hpipe.ev.begin() + nsub, g_hpipe.ev.begin() + 2 * nsub);
        for (int k = 0, c0 = 0; c0 < n; ++k, c0 += per) {
            const int nk = (n - c0 < per) ? n - c0 : per;
            cudaMemcpyAsync(dV + (size_t)c0 * M * M, A + (size_t)(b0 + c0) * M * M, mat * nk, cudaMemcpyHostToDevice, sH);
            cudaEventRecord(evH[k], sH);
        }
        cudaMemsetAsync(dinfo, 0, sizeof(int) * (size_t)n, sC);
        SyevHostCtx ctx{M, per, A + (size_t)b0 * M * M, w + (size_t)b0 * M, V + (size_t)b0 * M * M,
                        info ? info + b0 : nullptr, dV, dw, dinfo, sD, &evH, &evC};
        PassHooks hooks{syev_host_pre, syev_host_post, &ctx};
        rc = syev_pass(dV, M, n, dw, dV, dinfo, ws, sC, &hooks);     // in place
        launches += g_launches;
        // the arena is reused by the next pass: everything of this one must have left it
        cudaStreamSynchronize(sC);
        cudaStreamSynchronize(sD);
        cudaStreamSynchronize(sH);
    }
    cudaError_t ce = cudaGetLastError();
    if (rc == 0 && ce != cudaSuccess) rc = (int)ce;
    g_launches = launches;
    return rc;
}

// context of the copy hooks of letkf_analysis_batched_host: up to four output arrays
struct AnaHostCtx {
    int per, nout;
    char* host[4]; const char* dev[4]; size_t bytes[4];       // per grid point, at the start of the pass
    cudaStream_t sD;
    std::vector<cudaEvent_t>* evH;
    std::vector<cudaEvent_t>* evC;
};
static int ana_host_pre(void* c, int b0, int, cudaStream_t s)
{
    AnaHostCtx* x = static_cast<AnaHostCtx*>(c);
    return (int)cudaStreamWaitEvent(s, (*x->evH)[b0 / x->per], 0);
}
static int ana_host_post(void* c, int b0, int nk, cudaStream_t s)
{
    AnaHostCtx* x = static_cast<AnaHostCtx*>(c);
    cudaEvent_t e = (*x->evC)[b0 / x->per];
    cudaError_t ce;
    if ((ce = cudaEventRecord(e, s)) != cudaSuccess) return (int)ce;
    if ((ce = cudaStreamWaitEvent(x->sD, e, 0)) != cudaSuccess) return (int)ce;
    for (int q = 0; q < x->nout; ++q)
        if ((ce = cudaMemcpyAsync(x->host[q] + (size_t)b0 * x->bytes[q], x->dev[q] + (size_t)b0 * x->bytes[q],
                                  x->bytes[q] * (size_t)nk, cudaMemcpyDeviceToHost, x->sD)) != cudaSuccess) return (int)ce;
    return 0;
}

int letkf_analysis_batched_host(const double* Yb, const double* d, const double* rinv_loc,
                                const double* Xb, int M, int p, int nstate, int batch, double rho,
                                double* Xa, double* W, double* wbar, int* info)
{
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
    HostSubChunks max_sub_guard;
    // as letkf_syev_batched_host: one pass on the device at a time, inputs copied in sub-chunk by
    // sub-chunk, outputs read back as each sub-chunk's last kernel finishes
    const int chunk = syev_chunk(M, batch);
    const size_t sYb = sizeof(double) * (size_t)p * M, sd = sizeof(double) * (size_t)p;
    const size_t sX = sizeof(double) * (size_t)nstate * M, sW = sizeof(double) * (size_t)M * M;
    const size_t sw = sizeof(double) * (size_t)M;
    const size_t wsb = align_up(letkf_analysis_workspace_bytes(M, p, nstate, chunk), 256);
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
        int nsub, per;
        pass_partition(n, nsub, per);
        g_hpipe.events(2 * nsub);
        std::vector<cudaEvent_t> evH(g_hpipe.ev.begin(), g_hpipe.ev.begin() + nsub);
        std::vector<cudaEvent_t> evC(g_hpipe.ev.begin() + nsub, g_hpipe.ev.begin() + 2 * nsub);
        for (int k = 0, c0 = 0; c0 < n; ++k, c0 += per) {
            const int nk = (n - c0 < per) ? n - c0 : per;
            const size_t g0 = (size_t)(b0 + c0);
            if (p > 0) {
                cudaMemcpyAsync(dYb + (size_t)c0 * p * M, Yb + g0 * p * M, sYb * nk, cudaMemcpyHostToDevice, sH);
                cudaMemcpyAsync(dd + (size_t)c0 * p, d + g0 * p, sd * nk, cudaMemcpyHostToDevice, sH);
                cudaMemcpyAsync(dr + (size_t)c0 * p, rinv_loc + g0 * p, sd * nk, cudaMemcpyHostToDevice, sH);
            }
            cudaMemcpyAsync(dX + (size_t)c0 * nstate * M, Xb + g0 * nstate * M, sX * nk, cudaMemcpyHostToDevice, sH);
            cudaEventRecord(evH[k], sH);
        }
        cudaMemsetAsync(dinfo, 0, sizeof(int) * (size_t)n, sC);
        AnaHostCtx ctx;
        ctx.per = per; ctx.sD = sD; ctx.evH = &evH; ctx.evC = &evC; ctx.nout = 0;
        auto add = [&](void* h, const void* dv, size_t bytes) {
            ctx.host[ctx.nout] = static_cast<char*>(h); ctx.dev[ctx.nout] = static_cast<const char*>(dv);
            ctx.bytes[ctx.nout] = bytes; ++ctx.nout;
        };
        add(Xa + (size_t)b0 * nstate * M, dX, sX);
        if (W) add(W + (size_t)b0 * M * M, dW, sW);
        if (wbar) add(wbar + (size_t)b0 * M, dwb, sw);
        if (info) add(info + b0, dinfo, sizeof(int));
        PassHooks hooks{ana_host_pre, ana_host_post, &ctx};
        g_analysis_hooks = &hooks;
        rc = letkf_analysis_batched(dYb, dd, dr, dX, M, p, nstate, n, rho, dX, dW, dwb, dinfo, dwork, wsb, sC);
        g_analysis_hooks = nullptr;
        launches += g_launches;
        cudaStreamSynchronize(sC);
        cudaStreamSynchronize(sD);
        cudaStreamSynchronize(sH);
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
    HostSubChunks max_sub_guard;
    // The observation fields (V Ny Nx (M+1) doubles: 17 MB at 128 x 128 x 2 x 64) go in first, whole;
    // the background ensemble follows sub-chunk by sub-chunk and the analysis ensemble comes back
    // the same way (hooks as in letkf_analysis_batched_host).
    const int batch = Ny * Nx;
    const size_t nobs = (size_t)V * batch;
    const size_t sX = sizeof(double) * (size_t)nstate * M, sw = sizeof(double) * (size_t)M;
    const size_t wsb = align_up(letkf_analysis_grid_workspace_bytes(M, V, Ny, Nx, hw, nstate), 256);
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
    const int chunk = syev_chunk(M, batch);
    if (chunk < batch) return -8;                      // one pass only (180 GB: > 10^6 points at M = 64)
    int nsub, per;
    pass_partition(batch, nsub, per);
    g_hpipe.events(2 * nsub + 1);
    std::vector<cudaEvent_t> evH(g_hpipe.ev.begin(), g_hpipe.ev.begin() + nsub);
    std::vector<cudaEvent_t> evC(g_hpipe.ev.begin() + nsub, g_hpipe.ev.begin() + 2 * nsub);
    cudaEvent_t evF = g_hpipe.ev[2 * nsub];
    cudaMemcpyAsync(dYf, Yf, sizes[0], cudaMemcpyHostToDevice, sH);
    cudaMemcpyAsync(dyo, yo, sizes[1], cudaMemcpyHostToDevice, sH);
    if (obs_mask) cudaMemcpyAsync(dmask, obs_mask, sizes[2], cudaMemcpyHostToDevice, sH);
    cudaEventRecord(evF, sH);
    for (int k = 0, c0 = 0; c0 < batch; ++k, c0 += per) {
        const int nk = (batch - c0 < per) ? batch - c0 : per;
        cudaMemcpyAsync(dX + (size_t)c0 * nstate * M, Xb + (size_t)c0 * nstate * M, sX * nk, cudaMemcpyHostToDevice, sH);
        cudaEventRecord(evH[k], sH);
    }
    cudaStreamWaitEvent(sC, evF, 0);                   // the fields before anything is gathered
    cudaMemsetAsync(dinfo, 0, sizeof(int) * (size_t)batch, sC);
    AnaHostCtx ctx;
    ctx.per = per; ctx.sD = sD; ctx.evH = &evH; ctx.evC = &evC; ctx.nout = 0;
    auto add = [&](void* h, const void* dv, size_t bytes) {
        ctx.host[ctx.nout] = static_cast<char*>(h); ctx.dev[ctx.nout] = static_cast<const char*>(dv);
        ctx.bytes[ctx.nout] = bytes; ++ctx.nout;
    };
    add(Xa, dX, sX);
    if (wbar) add(wbar, dwb, sw);
    if (info) add(info, dinfo, sizeof(int));
    PassHooks hooks{ana_host_pre, ana_host_post, &ctx};
    g_analysis_hooks = &hooks;
    rc = letkf_analysis_grid(dYf, dyo, dmask, dX, M, V, Ny, Nx, nstate, hw, loc_kind, loc_scale, sigma_o, rho,
                             dX, dwb, dinfo, dwork, wsb, sC);
    g_analysis_hooks = nullptr;
    const int launches = g_launches;
    cudaStreamSynchronize(sC);
    cudaStreamSynchronize(sD);
    cudaStreamSynchronize(sH);
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
    if (strcmp(name, "force_generic") == 0) { g_force_generic = value != 0; return LETKF_OK; }
    if (strcmp(name, "pipeline") == 0) { g_pipeline = value != 0; return LETKF_OK; }
    if (strcmp(name, "sub_chunks") == 0) { g_max_sub = (value >= 1 && value <= PIPE_MAX_SUB) ? value : 8; return LETKF_OK; }
    if (strcmp(name, "mid_reg") == 0) { g_mid_reg = (value >= 0 && value <= 2) ? value : 1; return LETKF_OK; }
    if (strcmp(name, "split") == 0) { g_split = value != 0; return LETKF_OK; }
    if (strcmp(name, "log_shrink") == 0) { g_log_shrink = value >= 1 ? value : 1; return LETKF_OK; }
    if (strcmp(name, "ql_tpb") == 0) { g_ql_tpb = (value == 32 || value == 64 || value == 96) ? value : 0; return LETKF_OK; }
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

const char* letkf_status_string(int status)
{
    static thread_local char buf[96];
    if (status == 0) return "ok";
    if (status < 0) {
        snprintf(buf, sizeof(buf), "invalid argument %d (1-based position in the call)", -status);
        return buf;
    }
    return cudaGetErrorString((cudaError_t)status);
}

int letkf_version(void) { return LETKF_VERSION; }

}  // extern "C"

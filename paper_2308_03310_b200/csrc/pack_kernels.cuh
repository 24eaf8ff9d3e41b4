// pack_kernels.cuh -- M <= 16: TWO matrices per warp (section III: "when 1 < M < 32,
// 32/T batches are assigned to a single warp", T = 2^ceil(log2 M)).
//
// fast_tridiag<16> / fast_apply<16> give a matrix a whole warp: half the lanes hold no row, and ncu
// shows both kernels ISSUE bound at M = 16 (issue slots 71% / 56% busy, 4400 / 2800 warp instructions per
// matrix).  Here lanes 0-15 of a warp hold the rows (columns) of one matrix and lanes 16-31 those of
// the next, so every warp instruction works for two matrices.  The device functions are those of
// fast_kernels.cuh with j = lane % 16 and a TriShared per half warp: the shuffle trees of MT = 16 have
// four levels (they never leave the half warp), every barrier is a __syncwarp, a CTA is PK_WARPS
// independent warps.  The records in the workspace ((d, e), reflectors, flags) are those of the
// one-matrix-per-warp kernels, so ql_log_kernel / bisect_classify_kernel run unchanged in between.
// The two halves of a warp may take different routes through the apply kernel (eigenvectors of T by
// twisted factorisations / replay of logged rotations / the classic iteration): every phase is
// entered by the whole warp when either half needs it, with the other half predicated off.
// EVD only (letkf_syev_batched, fp64, reflector form); the analysis and fp32 calls keep one matrix per warp.
#pragma once
#include "fast_kernels.cuh"

namespace letkf {

constexpr int PK_WARPS = 4;                                  // warps per CTA: 8 matrices
constexpr int PK_LD = 17;                                    // padded stride of a 16 x 16 tile
constexpr int PK_REGION = RefLayout<16>::REGION;             // 272 = 16 x 17: staging tile, later the reflectors (192)
// doubles per half warp; 8 * PK_TRI_HALF = 64 (mod 128): the 16-byte broadcasts of the two halves of
// a warp come from different banks
constexpr int PK_TRI_HALF = PK_REGION + 5 * 16 + 8 + 32;     // + xs, v, p, pv, taus; red; (d, e) sink of an empty half
constexpr size_t pack16_tridiag_smem() { return sizeof(double) * 2 * PK_WARPS * PK_TRI_HALF; }

__global__ void __launch_bounds__(32 * PK_WARPS)
pack16_tridiag(const double* __restrict__ A_, Workspace ws, int M, int nbatch)
{
    constexpr int MT = 16;
    extern __shared__ __align__(16) double pk_sm[];
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5, h = lane >> 4, j = lane & 15;
    const long first = ((long)blockIdx.x * PK_WARPS + wp) * 2;
    if (first >= nbatch) return;                             // (whole warp; the kernel has no block barrier)
    const bool live = first + h < nbatch;                    // odd batch: the last half warp repeats the last matrix, stores nothing
    const size_t b = live ? (size_t)(first + h) : (size_t)(nbatch - 1);
    double* base = pk_sm + (size_t)(wp * 2 + h) * PK_TRI_HALF;
    double* tile = base;
    double* small = base + PK_REGION;
    TriShared<double> sh;
    sh.Rf = base;
    sh.xs = small; sh.vbuf = small + 16; sh.pbuf = small + 32; sh.pv = small + 48; sh.taus = small + 64; sh.red = small + 80;
    double* dws = live ? ws.dws + b * M : small + 88;
    double* ews = live ? ws.ews + b * M : small + 104;

    // a_j[c] = A[max(j,c)][min(j,c)] (only the lower triangle is read)
    const double* Ab = A_ + b * M * M;
    if (j < M) {
        int r = 0;
        for (; r + 8 <= M; r += 8) {
            double tmp[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) tmp[u] = Ab[(r + u) * M + j];
#pragma unroll
            for (int u = 0; u < 8; ++u) tile[(r + u) * PK_LD + j] = tmp[u];
        }
        for (; r < M; ++r) tile[r * PK_LD + j] = Ab[r * M + j];
    }
    __syncwarp();
    double a[MT];
#pragma unroll
    for (int c = 0; c < MT; ++c) {
        const int hi = max(j, c), lo = min(j, c);
        a[c] = (hi < M) ? tile[hi * PK_LD + lo] : 0.0;
    }
    __syncwarp();

    // prologue = the look-ahead of a fictitious pivot M (as in fast_tridiag)
    {
        const int i0 = M - 1;
        const double x = pick<MT>(a, i0);
        if (j == i0) dws[i0] = x;
        sh.xs[j] = (j < i0 - 1) ? x : 0.0;
        if (j == i0 - 1) sh.red[4] = x;
        double part = (j < i0 - 1) ? x * x : 0.0;
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
        if (j == 0) { sh.red[0] = part; ews[M - 1] = 0.0; }
        __syncwarp();
    }
    pivot_groups_range<MT, 1, 0>(a, sh, M, dws, ews, j);
    __syncwarp();
    if (live) {
        double* out = ws.refl + b * ws.reflstride;
        for (int k = j; k < RefLayout<MT>::TOTAL; k += 16) out[k] = sh.Rf[k];
        out[RefLayout<MT>::TOTAL + j] = (j >= 1 && j <= M - 1) ? sh.taus[j] : 0.0;
        out[RefLayout<MT>::TOTAL + 16 + j] = 0.0;
    }
}

// doubles per half warp of pack16_apply: reflectors + taus [224], ds, es, wsrt [16 each], tile [272],
// inv, perm [16 ints each], ctl [4 ints]; 8 * PK_AP_HALF = 64 (mod 128)
constexpr int PK_AP_HALF = 224 + 48 + 272 + 16 + 2 + 6;
static_assert((PK_AP_HALF * 8) % 128 == 64 && PK_AP_HALF % 2 == 0 && (PK_TRI_HALF * 8) % 128 == 64, "bank offset of the second half");
constexpr size_t pack16_apply_smem() { return sizeof(double) * 2 * PK_WARPS * PK_AP_HALF; }

// reflectors i = 8G+1 ... min(8G+8, M-1) applied to the column held by this thread (q_group of
// fast_kernels.cuh without the shortcut for tau = 0: the halves of a warp stay in step)
template <int G>
__device__ __forceinline__ void pk_q_group(double (&q)[16], const double* Rf, const double* taus, int M)
{
#pragma unroll 1
    for (int i = 8 * G + 1; i <= 8 * G + 8 && i <= M - 1; ++i) {
        const double* v1 = Rf + RefLayout<16>::base(G) + (i - 1 - 8 * G) * RefLayout<16>::len(G);
        const double ns1 = -taus[i] * dot_blocks<16, G, true>(q, v1);
#pragma unroll
        for (int g = G; g >= 0; --g) { axpy_block<16>(q, v1, ns1, g); __syncwarp(); }
    }
}

__global__ void __launch_bounds__(32 * PK_WARPS)
pack16_apply(double* __restrict__ V_, double* __restrict__ w_, int* __restrict__ info_, Workspace ws, int M, int nbatch)
{
    constexpr int MT = 16;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(16) double pk_sm[];
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5, h = lane >> 4, j = lane & 15;
    const long first = ((long)blockIdx.x * PK_WARPS + wp) * 2;
    if (first >= nbatch) return;
    const bool live = first + h < nbatch;
    const size_t b = live ? (size_t)(first + h) : (size_t)(nbatch - 1);
    double* base = pk_sm + (size_t)(wp * 2 + h) * PK_AP_HALF;
    double* R = base;                                   // reflectors, RefLayout<16> order
    double* taus = R + RefLayout<MT>::TOTAL;
    double* ds = base + 224;
    double* es = ds + 16;
    double* wsrt = es + 16;
    double* tile = wsrt + 16;                           // [16][17]
    int* inv = reinterpret_cast<int*>(tile + 272);      // output column of QL-order column c
    int* perm = inv + 16;                               // position of the k-th smallest eigenvalue
    int* ctl = perm + 16;

    const int flag = ws.flags[b];
    const bool direct = flag == FLAG_GETVEC;
    const bool replay = flag == FLAG_REPLAY;
    {   // the reflectors fly in while the eigenvectors of T are formed
        const double* src = ws.refl + b * ws.reflstride;
        for (int k = 2 * j; k < refl_doubles<MT>(); k += 32) cp_async16(R + k, src + k);
    }
    ds[j] = (j < M) ? ws.dws[b * M + j] : 0.0;
    es[j] = (j < M - 1) ? ws.ews[b * M + j] : 0.0;
    const bool sorted = direct || replay;               // w and perm are the QL kernel's
    wsrt[j] = (sorted && j < M) ? w_[b * M + j] : 0.0;
    perm[j] = (sorted && j < M) ? ws.perm[b * M + j] : j;
    __syncwarp();
    inv[perm[j]] = j;
    __syncwarp();

    double z[MT];
    bool columns = false;                               // z holds an eigenvector of T rather than a row of Z
    bool slow = !direct && !replay;                     // FLAG_SLOW (rotation log unusable): classic QL below

    if (__any_sync(FULL, direct)) {
        // ---- eigenvectors of T by twisted factorisations (direct_eigenvectors of fast_kernels.cuh, per half warp)
        const double eps = 1.1102230246251565e-16;
        double nrm = (j < M) ? fabs(ds[j]) + (j < M - 1 ? fabs(es[j]) : 0.0) : 0.0;
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) nrm = fmax(nrm, __shfl_xor_sync(FULL, nrm, o));
        const double thr = eps * nrm;
        bool cut = true;
        if (j < M - 1) cut = fabs(es[j]) <= fmax(eps * (fabs(ds[j]) + fabs(ds[j + 1])), GV_SPLIT * thr);
        __syncwarp();
        if (cut) es[j] = 0.0;
        const unsigned cuts = (__ballot_sync(FULL, cut) >> (16 * h)) & 0xffffu;
        __syncwarp();
        int lo = 0, hi = M - 1;
        double lam = 0.0;
        if (j < M) {
            const unsigned below = cuts & ((1u << j) - 1u);
            lo = below ? 32 - __clz((int)below) : 0;
            const unsigned above = cuts >> j;
            hi = above ? j + __ffs((int)above) - 1 : M - 1;
            if (hi > M - 1) hi = M - 1;
            lam = wsrt[inv[j]];
        }
        const bool own = j < M && lo < hi;
        double res = getvec<MT>(z, ds, es, lam, lo, hi, fmax(thr * eps, 1e-300));
        if (!own) {
            res = 0.0;
#pragma unroll
            for (int c = 0; c < MT; ++c) z[c] = (c == j) ? 1.0 : 0.0;
        }
        const bool bad = !(res <= 64.0 * eps * nrm * sqrt((double)M));
        const bool ok = ((__ballot_sync(FULL, bad) >> (16 * h)) & 0xffffu) == 0u;
        if (direct) { columns = ok; slow = !ok; }
        // eigenvalues closer than GV_GAP ||T|| inside a block: first-order symmetric orthogonalisation
        const double gapabs = GV_GAP * nrm;
        PartnerList pl;                                                 // same-block eigenvalues within GV_GAP ||T|| (the classifier bounds them)
        if (own && columns) {
            const int s0 = inv[j];
            for (int t = 1; s0 - t >= 0 && lam - wsrt[s0 - t] < gapabs; ++t) {
                const int q = perm[s0 - t];
                if (q >= lo && q <= hi) pl.add(q);
            }
            for (int t = 1; s0 + t < M && wsrt[s0 + t] - lam < gapabs; ++t) {
                const int q = perm[s0 + t];
                if (q >= lo && q <= hi) pl.add(q);
            }
        }
        const int npw = __reduce_max_sync(FULL, pl.np);                    // the whole warp walks the longest list
        if (npw > 0) {
#pragma unroll
            for (int i = 0; i < MT; ++i) tile[j * PK_LD + i] = z[i];
            __syncwarp();
#pragma unroll 1
            for (int t = 0; t < npw; ++t) {
                const int q = pl.get(t);
                const bool act = t < pl.np;
                const double* vq = tile + (act ? q : 0) * PK_LD;
                double d0 = 0.0, d1 = 0.0;
#pragma unroll
                for (int i = 0; i + 1 < MT; i += 2) {
                    d0 = fma(z[i], vq[i], d0); d1 = fma(z[i + 1], vq[i + 1], d1);
                    if ((i & 7) == 6) __syncwarp();
                }
                const double hh = act ? -0.5 * (d0 + d1) : 0.0;
#pragma unroll
                for (int i = 0; i < MT; ++i) {
                    z[i] = fma(hh, vq[i], z[i]);
                    if ((i & 7) == 7) __syncwarp();
                }
            }
            __syncwarp();
        }
    }

    if (__any_sync(FULL, replay)) {
        // ---- thread j replays the logged rotations on row j of the identity, one sweep per round
        if (replay) {
#pragma unroll
            for (int c = 0; c < MT; ++c) z[c] = (c == j) ? 1.0 : 0.0;
        }
        const int nsw = replay ? ws.nsweeps[b] : 0;
        const int nmax = __reduce_max_sync(FULL, nsw);
        const double2* rot = ws.rot + b * ws.logcap;
        double2* cs = reinterpret_cast<double2*>(tile);                 // [16] by column, identity outside [lo, m)
        int spos = 0;
#pragma unroll 1
        for (int s = 0; s < nmax; ++s) {
            int lo = 0, m = 0;
            if (s < nsw) { const uint32_t hw = ws.hdr[b * ws.swcap + s]; lo = hw & 0xffff; m = hw >> 16; }
            __syncwarp();
            cs[j] = (j >= lo && j < m) ? rot[spos + (m - 1 - j)] : make_double2(1.0, 0.0);
            __syncwarp();
            if (s < nsw) apply_sweep<MT>(z, cs, lo, m);
            spos += m - lo;
        }
        __syncwarp();
    }

    if (__any_sync(FULL, slow)) {
        // ---- slow path (LETKF_INFO_SLOWPATH): the classic iteration, one sweep at a time; lane 0 of the
        // half runs the recurrences of ql_next_sweep, its 16 lanes apply the sweep to their rows
        double*  dsm  = tile;                                           // [16]
        double*  esm  = tile + 16;                                      // [16]
        double2* sink = reinterpret_cast<double2*>(tile + 32);          // [16] in generation order
        double2* csb  = sink + 16;                                      // [16] by column
        __syncwarp();
        if (slow) {
#pragma unroll
            for (int c = 0; c < MT; ++c) z[c] = (c == j) ? 1.0 : 0.0;
            dsm[j] = (j < M) ? ws.dws[b * M + j] : 0.0;
            esm[j] = (j < M) ? ws.ews[b * M + j] : 0.0;
        }
        __syncwarp();
        QLState st{0, 0, 0, 0.0};
        if (slow && j == 0) { esm[M - 1] = 0.0; st.thr = ql_threshold(dsm, esm, 1, M); }
        bool going = slow;
        for (;;) {
            if (going && j == 0) {
                int lo = 0, m = 0;
                ctl[0] = ql_next_sweep(st, dsm, esm, 1, M, sink, M, lo, m);
                ctl[1] = lo; ctl[2] = m;
            }
            __syncwarp();
            if (going && ctl[0] != 1) going = false;
            if (!__any_sync(FULL, going)) break;
            int lo = 0, m = 0;
            if (going) { lo = ctl[1]; m = ctl[2]; csb[j] = (j >= lo && j < m) ? sink[m - 1 - j] : make_double2(1.0, 0.0); }
            __syncwarp();
            if (going) apply_sweep<MT>(z, csb, lo, m);
            __syncwarp();
        }
        int* permsm = reinterpret_cast<int*>(sink);                     // the sink is free now
        if (slow && j == 0) { sort_eigenvalues(dsm, 1, permsm, 1, M); ctl[3] = st.fail; }
        __syncwarp();
        if (slow) {
            if (j < M) { inv[permsm[j]] = j; if (live) w_[b * M + j] = dsm[j]; }
            if (j == 0 && info_ && live) info_[b] = ctl[3] | 0x40000000;
        }
        __syncwarp();
    }

    cp_async_wait_all();
    __syncwarp();
    // rows of Z -> eigenvectors of T (thread k holds column k, QL order)
    if (__any_sync(FULL, !columns)) {
        if (!columns) {
#pragma unroll
            for (int c = 0; c < MT; ++c) tile[j * PK_LD + c] = z[c];
        }
        __syncwarp();
        if (!columns) {
#pragma unroll
            for (int rr = 0; rr < MT; ++rr) z[rr] = tile[rr * PK_LD + j];
        }
        __syncwarp();
    }
    // V = H_{M-1} ... H_1 Z
    pk_q_group<0>(z, R, taus, M);
    pk_q_group<1>(z, R, taus, M);
    // sorted, row-major V through the tile: thread k scatters its column into output column inv[k],
    // thread t then writes column t of every row (128 contiguous bytes per row and half warp)
    __syncwarp();
    if (j < M) {
        const int oc = inv[j];
#pragma unroll
        for (int rr = 0; rr < MT; ++rr) tile[rr * PK_LD + oc] = z[rr];
    }
    __syncwarp();
    if (live && j < M) {
        double* V = V_ + b * M * M;
#pragma unroll 8
        for (int rr = 0; rr < M; ++rr) V[rr * M + j] = tile[rr * PK_LD + j];
    }
}

}  // namespace letkf

// bisect_kernel.cuh -- step a4 for the LATENCY regime (with 64
// GPUs the paper's share is 256 matrices per GPU, "too small for the batched EVD").
//
// The QL iteration of ql_kernel.cuh is one thread walking ~1.05 M^2 dependent rotation steps per
// matrix: 0.45 ms at M = 64 however few matrices there are.  A small batch leaves the machine empty,
// so here a matrix gets M THREADS for its eigenvalues instead of one: thread k finds the eigenvalue
// with index k - lo of the unreduced block [lo, hi] of T that contains position k by multisection on
// the Sturm count (number of negative pivots of T - x I = number of eigenvalues below x; three
// interior points per round, i.e. three independent recurrences in flight and a factor 4 per round:
// ~29 rounds of <= M steps against ~4300 dependent steps).  The eigenvalues are then sorted and the
// matrix classified exactly as ql_log_kernel does in QL_CLASSIFY mode (common.cuh, GV_*): the apply
// kernel forms the eigenvectors of T itself (FLAG_GETVEC), or the logging QL pass follows
// (FLAG_PENDING, shifted by these eigenvalues).  Same splitting criterion, same outputs (w ascending,
// perm, s1 by position), so everything downstream is unchanged.
#pragma once
#include "common.cuh"
#include "fast_kernels.cuh"

namespace letkf {

// Sturm counts of T[lo..hi] - x I at three points at once: number of negative pivots of L D L^T.
// e2[i] = e_i^2 (coupling i, i+1); a pivot smaller than pivmin in magnitude counts as -pivmin.
__device__ __forceinline__ void sturm3(const double* ds, const double* e2, int lo, int hi, double pivmin,
                                       double x1, double x2, double x3, int& c1, int& c2, int& c3)
{
    double q1 = ds[lo] - x1, q2 = ds[lo] - x2, q3 = ds[lo] - x3;
    int n1 = 0, n2 = 0, n3 = 0;
    for (int i = lo;; ++i) {
        q1 = (fabs(q1) < pivmin) ? -pivmin : q1;
        q2 = (fabs(q2) < pivmin) ? -pivmin : q2;
        q3 = (fabs(q3) < pivmin) ? -pivmin : q3;
        n1 += q1 < 0.0 ? 1 : 0;
        n2 += q2 < 0.0 ? 1 : 0;
        n3 += q3 < 0.0 ? 1 : 0;
        if (i == hi) break;
        const double ee = e2[i], dn = ds[i + 1];
        q1 = fma(-ee, fast_rcp(q1), dn - x1);
        q2 = fma(-ee, fast_rcp(q2), dn - x2);
        q3 = fma(-ee, fast_rcp(q3), dn - x3);
    }
    c1 = n1; c2 = n2; c3 = n3;
}

template <int MT>
__global__ void __launch_bounds__(FastCfg<MT>::NT)
bisect_classify_kernel(Workspace ws, int M, double* __restrict__ w, int* __restrict__ info)
{
    using C = FastCfg<MT>;
    __shared__ double ds[MT], es[MT], e2[MT], lam[MT], wsrt[MT];
    __shared__ short blk_s[MT];                           // block of the k-th smallest eigenvalue (negated: 1 x 1 block)
    __shared__ unsigned cutw[2];
    const int k = threadIdx.x;
    const size_t b = blockIdx.x;
    if (k < MT) {
        ds[k] = (k < M) ? ws.dws[b * M + k] : 0.0;
        es[k] = (k < M - 1) ? ws.ews[b * M + k] : 0.0;
    }
    __syncthreads();
    // the threshold and the split of ql_log_kernel / fast_apply, on the same numbers
    const double eps = 1.1102230246251565e-16;
    double nrm = 0.0;
    for (int i = 0; i < M; ++i) nrm = fmax(nrm, fabs(ds[i]) + (i < M - 1 ? fabs(es[i]) : 0.0));
    const double thr = eps * nrm;
    bool cut = true;
    if (k < M - 1) cut = fabs(es[k]) <= fmax(eps * (fabs(ds[k]) + fabs(ds[k + 1])), GV_SPLIT * thr);
    __syncthreads();
    if (k < MT) { const double ev = cut ? 0.0 : es[k]; es[k] = ev; e2[k] = ev * ev; }
    const unsigned cw = __ballot_sync(0xffffffffu, cut);
    if ((k & 31) == 0) cutw[k >> 5] = cw;
    __syncthreads();
    const unsigned long long cuts = (C::NW > 1) ? ((unsigned long long)cutw[1] << 32 | cutw[0]) : (unsigned long long)cutw[0];
    int lo = 0, hi = M - 1;
    if (k < M) {
        const unsigned long long below = cuts & ((1ull << k) - 1ull);
        lo = below ? 64 - __clzll((long long)below) : 0;
        const unsigned long long above = cuts >> k;
        hi = above ? k + __ffsll((long long)above) - 1 : M - 1;
        if (hi > M - 1) hi = M - 1;
    }
    double lk = 0.0;
    if (k < M) {
        if (lo == hi) {
            lk = ds[k];
        } else {
            // Gershgorin interval of the block, widened by the rounding of the counts
            double gl = 1.7976931348623157e308, gu = -1.7976931348623157e308;
            for (int i = lo; i <= hi; ++i) {
                const double rad = (i > lo ? fabs(es[i - 1]) : 0.0) + (i < hi ? fabs(es[i]) : 0.0);
                gl = fmin(gl, ds[i] - rad);
                gu = fmax(gu, ds[i] + rad);
            }
            const double pivmin = fmax(thr * eps, 1e-300);
            const double widen = 2.0 * thr * (double)(hi - lo + 1) + 2.0 * pivmin;
            double a = gl - widen, c = gu + widen;            // count(a) = 0 <= j < n = count(c)
            const int j = k - lo;
            for (int round = 0; round < 64; ++round) {
                const double wdt = c - a;
                if (!(wdt > fmax(2.0 * eps * fmax(fabs(a), fabs(c)), 0.125 * thr))) break;
                const double x2 = a + 0.5 * wdt, x1 = a + 0.25 * wdt, x3 = a + 0.75 * wdt;
                int c1, c2, c3;
                sturm3(ds, e2, lo, hi, pivmin, x1, x2, x3, c1, c2, c3);
                // eigenvalue j (0-based) lies in the first sub-interval whose upper count exceeds j
                if (j < c1) c = x1;
                else if (j < c2) { a = x1; c = x2; }
                else if (j < c3) { a = x2; c = x3; }
                else a = x3;
            }
            lk = a + 0.5 * (c - a);
        }
        lam[k] = lk;
    }
    __syncthreads();
    // sort by rank, classify (as the tail of ql_log_kernel in QL_CLASSIFY mode)
    int rank = 0;
    if (k < M) {
        for (int jj = 0; jj < M; ++jj) {
            const double u = lam[jj];
            rank += (u < lk || (u == lk && jj < k)) ? 1 : 0;
        }
        w[b * M + rank] = lk;
        ws.perm[b * M + rank] = k;
        ws.s1[b * M + k] = lk;
        wsrt[rank] = lk;
        blk_s[rank] = (short)((lo == hi) ? -(lo + 1) : (lo + 1));
    }
    __syncthreads();
    bool hard = false;
    if (k + 1 < M) hard = gv_hard_at(k, M, nrm, [&](int u) { return wsrt[u]; }, [&](int u) { return (int)blk_s[u]; });
    const int anyhard = __syncthreads_or(hard ? 1 : 0);
    if (k == 0) {
        ws.nsweeps[b] = 0;
        ws.flags[b] = anyhard ? FLAG_PENDING : FLAG_GETVEC;
        if (info) info[b] = 0;
        if (ws.rot_counter && !anyhard) atomicAdd(ws.rot_counter + 1, 1ull);
    }
}

}  // namespace letkf

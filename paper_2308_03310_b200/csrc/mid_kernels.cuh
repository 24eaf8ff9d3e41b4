// mid_kernels.cuh -- 64 < M <= 160: the matrix no longer fits the registers of two warps, but it
// still fits ONE SM's shared memory (M (M+1) doubles: 74 KB at M = 96, 132 KB at M = 128, 206 KB
// at M = 160).  One CTA of ceil32(M) threads per matrix, thread j = row j, the matrix resident in
// shared memory for the whole kernel (one HBM round trip per kernel, as on the register path);
// the any-M kernels of generic_kernels.cuh, which keep the matrix in global memory / L2, remain
// for M > 160 (BASELINE config 5: "from M = 128 up ... forces a blocked or tiled strategy").
//
//   mid_tridiag_formq   a3 + explicit Q^T (Householder), same conventions as
//                       generic_tridiag_formq: pivots i = M-1 ... 1, H_i acts on 0..i-1,
//                       V receives Q^T ("Qt" layout: Qt[c][r] = Q[r][c])
//   mid_apply           a5: replay of the rotation log on the columns of Q (rows of Q^T),
//                       eigenvalue sort, row-major V out
// The row stride M+1 is odd, so "same column, 32 consecutive rows" and "same row, consecutive
// columns" are both conflict-free for 8-byte accesses.
#pragma once
#include "common.cuh"

namespace letkf {

static inline bool mid_supported(int M) { return M > 64 && M <= 160; }
static inline int mid_threads(int M) { return (M + 31) / 32 * 32; }
// row stride of the resident matrix: >= M+1 and = 2 (mod 16) doubles, so that a row can be read
// with 16-byte loads (even) and the 8 lanes of a quarter warp, one row each, hit 8 x 4 different
// banks (stride = 4 words mod 32)
__host__ __device__ inline int mid_ld(int M) { return ((M + 1 + 13) / 16) * 16 + 2; }
constexpr int MID_TPR = 4;     // threads per row in mid_tridiag_formq
static inline size_t mid_tridiag_smem(int M)
{
    return sizeof(double) * ((size_t)M * mid_ld(M) + 3 * ((size_t)mid_ld(M)) + (size_t)MID_TPR * mid_threads(M) + 64 + 8);
}
// the columns of a matrix are dealt to this many CTAs (a cluster) in mid_apply
static inline int mid_apply_split(int M) { return (M > 96 && M <= 128) ? 2 : 1; }
static inline int mid_apply_cols(int M) { const int ns = mid_apply_split(M); return ((M + ns - 1) / ns + 1) & ~1; }
static inline size_t mid_apply_smem(int M, int swcap, int ms)
{
    const int ld = (mid_apply_cols(M) + 1) | 1;
    return sizeof(double) * ((((size_t)M * ld + 1) & ~(size_t)1) + 4 * (size_t)ms * (size_t)M) + sizeof(uint32_t) * (size_t)swcap + sizeof(int) * (size_t)M + 32;
}
// sweeps staged per barrier round of mid_apply: as many (<= 4) as shared memory holds beside the
// matrix -- beside three CTAs per SM when the columns are split
static inline int mid_apply_round(int M, int swcap)
{
    const size_t cap = mid_apply_split(M) > 1 ? (size_t)(228 * 1024) / 3 - 1024 : (size_t)226 * 1024;
    int ms = 4;
    while (ms > 1 && mid_apply_smem(M, swcap, ms) > cap) ms >>= 1;
    return ms;
}

// Block-wide sum for a run-time number of warps (<= 20); ONE barrier: consecutive calls alternate
// between two scratch rows (`which`), so a warp that runs ahead into the next call cannot
// overwrite partial sums that a slower warp is still reading.  All threads get the result.
__device__ __forceinline__ double mid_block_sum(double v, double* red, int nwarps, int which)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* row = red + which * 32;
    v = warp_sum(v);
    if (lane == 0) row[warp] = v;
    __syncthreads();
    double t = 0.0;
    for (int w = 0; w < nwarps; ++w) t += row[w];
    return t;
}

// Explicit Q^T = H_1 H_2 ... H_{M-1} (H_i acts on indices 0..i-1) row by row: row j of Q^T is
// e_j^T H_{j+1} ... H_{M-1}, so the rows do not depend on each other and a row never has to live
// in shared memory: 8 lanes hold one row in registers (lane h owns the column pairs h, h+8, ...:
// 16-byte broadcast loads of the reflectors, which stay where the reduction left them: row i of S,
// zero-padded to a multiple of 16 columns), apply every reflector to it (dot product reduced
// with three shuffles, no barrier) and store it straight to global memory.  Row j costs
// sum_{i>j} 4i flops, so a group takes row g and then row M-1-g: all warps stay busy to the end.
template <int MT, bool KEEPV>
__device__ __forceinline__ void mid_formq_rows(const double* S, int LD, const double* taus, int M, double* Qt)
{
    constexpr int NP = MT / 16;                       // column pairs per lane
    const int tid = threadIdx.x, h = tid & 7, g = tid >> 3, ngrp = blockDim.x >> 3;
    const int g0 = g & ~3;                            // first group of this warp
    const double2* S2 = reinterpret_cast<const double2*>(S);
    const int LD2 = LD >> 1;
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
        const int j = pass == 0 ? g : M - 1 - g;
        const bool valid = pass == 0 ? (j < M) : (j >= ngrp);
        const int jmin = pass == 0 ? g0 : max(M - 1 - (g0 + 3), 0);    // smallest row of the warp
        if (pass == 1 && M - 1 - g0 < ngrp) continue;                  // no valid row in this warp
        double2 x[NP];
#pragma unroll
        for (int k = 0; k < NP; ++k) {
            const int c = 2 * h + 16 * k;
            x[k] = make_double2((valid && c == j) ? 1.0 : 0.0, (valid && c + 1 == j) ? 1.0 : 0.0);
        }
#pragma unroll 1
        for (int i = jmin + 1; i <= M - 1; ++i) {
            const double tau = taus[i];
            if (tau == 0.0) continue;
            const double2* v2 = S2 + (size_t)i * LD2 + h;
            double a0 = 0.0, a1 = 0.0;
            double2 v[NP];
#pragma unroll
            for (int k = 0; k < NP; ++k) {
                if (16 * k < i) {
                    v[k] = v2[8 * k];
                    a0 = fma(x[k].x, v[k].x, a0);
                    a1 = fma(x[k].y, v[k].y, a1);
                }
            }
            double acc = a0 + a1;
            acc += __shfl_xor_sync(0xffffffffu, acc, 1);
            acc += __shfl_xor_sync(0xffffffffu, acc, 2);
            acc += __shfl_xor_sync(0xffffffffu, acc, 4);
            acc *= -tau;
#pragma unroll
            for (int k = 0; k < NP; ++k) {
                if (16 * k < i) {
                    const double2 u = KEEPV ? v[k] : v2[8 * k];
                    x[k].x = fma(acc, u.x, x[k].x);
                    x[k].y = fma(acc, u.y, x[k].y);
                }
            }
        }
        if (valid) {
            double* qrow = Qt + (size_t)j * M;
#pragma unroll
            for (int k = 0; k < NP; ++k) {
                const int c = 2 * h + 16 * k;
                if ((M & 1) == 0) {
                    if (c < M) *reinterpret_cast<double2*>(qrow + c) = x[k];
                } else {
                    if (c < M) qrow[c] = x[k].x;
                    if (c + 1 < M) qrow[c + 1] = x[k].y;
                }
            }
        }
    }
}

// MID_TPR threads per row: thread (j, h) = (tid % RP, tid / RP), RP = ceil32(M), owns the column
// pairs p = h, h + TPR, ... of row j (16-byte accesses); the partial products of a row meet in
// shared memory.  vs / wsm are kept zero at index i (the first dead column) so that a pair that
// straddles the active range contributes nothing.
template <int MT>
__global__ void __launch_bounds__(MT * MID_TPR, MT == 96 ? 2 : 1)
mid_tridiag_formq(const double* __restrict__ A_, double* V_, Workspace ws, int M)
{
    extern __shared__ __align__(16) double sm[];
    const int LD = mid_ld(M);
    constexpr int RP = MT;
    double* S    = sm;                       // [M][LD]
    double* vs   = sm + (size_t)M * LD;      // [LD]
    double* wsm  = vs + LD;                  // [LD]
    double* taus = wsm + LD;                 // [LD]
    double* pd   = taus + LD;                // [TPR][RP] partial products
    double* red  = pd + MID_TPR * RP;        // [2][32]
    const int tid = threadIdx.x, j = tid % RP, h = tid / RP, nw = blockDim.x >> 5;
    const size_t b = blockIdx.x;
    const double* A = A_ + b * M * M;
    double* dws = ws.dws + b * M;
    double* ews = ws.ews + b * M;

    // full symmetric copy of the lower triangle: thread (j, h) copies column j of rows h, h+TPR, ...
    if (j < M) {
        for (int r = h; r < M; r += MID_TPR) {
            const double val = (r >= j) ? A[(size_t)r * M + j] : A[(size_t)j * M + r];
            S[r * LD + j] = val;
        }
    }
    for (int c = tid; c < LD; c += blockDim.x) { vs[c] = 0.0; wsm[c] = 0.0; }
    __syncthreads();

    const double2* row2 = reinterpret_cast<const double2*>(S + (size_t)j * LD);
    double2* row2w = reinterpret_cast<double2*>(S + (size_t)j * LD);
    const double2* v2 = reinterpret_cast<const double2*>(vs);
    const double2* w2 = reinterpret_cast<const double2*>(wsm);

    for (int i = M - 1; i >= 1; --i) {
        const double xj = (j < i) ? S[j * LD + i] : 0.0;
        const double sigma = mid_block_sum((h == 0 && j < i - 1) ? xj * xj : 0.0, red, nw, 0);
        const double alpha = S[(i - 1) * LD + i];
        double tau = 0.0, scal = 0.0, beta = alpha;                // sigma == 0: H_i = I (reading G19)
        if (sigma != 0.0) {
            const double nrm2 = fma(alpha, alpha, sigma);
            const double rinv = rsqrt(nrm2);
            beta = -copysign(nrm2 * rinv, alpha);
            tau = fma(fabs(alpha), rinv, 1.0);
            scal = 1.0 / (alpha - beta);
        }
        const double vj = (j < i - 1) ? xj * scal : ((j == i - 1) ? 1.0 : 0.0);
        if (h == 0) {
            if (j <= i && j < M) vs[j] = vj;                       // vs[i] = 0
            if (j == i) dws[i] = S[i * LD + i];
            if (j == 0) { ews[i - 1] = beta; taus[i] = tau; }
        }
        __syncthreads();
        const int npair = (i + 1) >> 1;
        if (tau != 0.0) {
            double a0 = 0.0, a1 = 0.0;
            if (j < i) {
#pragma unroll 4
                for (int p = h; p < npair; p += MID_TPR) {
                    const double2 r = row2[p], v = v2[p];
                    a0 = fma(r.x, v.x, a0);
                    a1 = fma(r.y, v.y, a1);
                }
            }
            pd[h * RP + j] = a0 + a1;
            __syncthreads();
            double pj = 0.0;
            if (j < i) {
#pragma unroll
                for (int hh = 0; hh < MID_TPR; ++hh) pj += pd[hh * RP + j];
                pj *= tau;
            }
            const double ptv = mid_block_sum(h == 0 ? pj * vj : 0.0, red, nw, 1);
            const double wj = pj - (0.5 * tau * ptv) * vj;        // w = p - (tau/2)(p.v) v
            if (h == 0 && j <= i && j < M) wsm[j] = (j < i) ? wj : 0.0;
            __syncthreads();
            if (j < i) {                                           // S11 -= v w^T + w v^T
#pragma unroll 4
                for (int p = h; p < npair; p += MID_TPR) {
                    double2 r = row2w[p];
                    const double2 v = v2[p], w = w2[p];
                    r.x = fma(-vj, w.x, fma(-wj, v.x, r.x));
                    r.y = fma(-vj, w.y, fma(-wj, v.y, r.y));
                    row2w[p] = r;
                }
            }
        }
        if (h == 0 && j < i) S[i * LD + j] = vj;                   // keep the reflector in the dead row i (no
        if (h == 1 && j < 16 && i + j < LD) S[i * LD + i + j] = 0.0;  // update touches it), zero-padded for mid_formq_rows
        __syncthreads();
    }
    if (tid == 0) { dws[0] = S[0]; ews[M - 1] = 0.0; }

    __syncthreads();                                               // taus, reflector rows complete
    double* Qt = V_ + b * M * M;
    mid_formq_rows<MT, MT <= 128>(S, LD, taus, M, Qt);
}

// a3 with the matrix in REGISTERS (the idea of fast_tridiag_formq with four threads per row): the
// shared-memory copy of A is only the staging area of the load; from then on thread (j, h) =
// (tid % MT, tid / MT) holds the column pairs h, h+4, ... of row j, and shared memory carries
// nothing but the vectors every row needs: v_i (written, zero-padded, into row i of S, where the
// explicit-Q pass finds it) and p.  h is the same in all lanes of a warp, so a 16-byte load of
// (v_c, v_c+1) is ONE broadcast wavefront that feeds two FMAs in every lane (with the four
// threads of a row in one warp the same load is four wavefronts and the shared-memory pipe
// binds: measured, 1.3 / 1.7 k cycles per pivot for the product / the update at M = 96).  Pivot i:
//   B0  the raw row i (final: its four owners dumped it after pivot i+1's update) is in xs
//       -> warps of h = 0: sigma, tau, beta, v_i into row i of S
//   B1  -> partial products sum_c a_jc v_c over the thread's pairs (8-column blocks with 8k < i:
//          block-uniform bounds, static register indices) into pd[h][j]
//   B2  -> warps of h = 0: p_j = tau sum_h pd[h][j], the warp's share of p.v
//   B3  -> a_jc -= v_j p_c + (p_j - tau (p.v) v_j) v_c
// HEAD (64 < M <= 128, option mid_split): the kernel stops after pivot 64 and hands the trailing 64 x 64
// block to the register kernels of fast_kernels.cuh (fast_tridiag<64> + fast_tridiag_tail: a pivot there
// costs ~2400 cycles in 64 threads against ~3300 here in 4 ceil32(M)) -- 63 of the M - 1 pivots.  It leaves
// the block as a dense 64 x 64 matrix in blk[b], (d_i, e_{i-1}) for i >= 64, and its reflectors (rows
// 64 ... M-1 of S) and taus behind the RefLayout<64> record of ws.refl; mid_formq_split then gathers both
// sets of reflectors and forms Q^T as before.
__host__ __device__ inline int mid_split_fast_doubles() { return 32 * 8 * 9 + 64; }      // RefLayout<64>::TOTAL + 64 taus
static inline int mid_split_refl_doubles(int M) { return mid_split_fast_doubles() + (M - 64 + 1) * mid_ld(M); }
template <int MT, bool HEAD = false>
__global__ void __launch_bounds__(MT * MID_TPR, MT == 96 ? 2 : 1)
mid_tridiag_formq_reg(const double* __restrict__ A_, double* V_, Workspace ws, int M)
{
    double* blk = reinterpret_cast<double*>(ws.rot);      // HEAD: the trailing blocks [n][64][64], flat in the (still unused) log area
    extern __shared__ __align__(16) double sm[];
    static_assert(MID_TPR == 4, "column pairs are dealt to four threads per row");
    constexpr int NP = MT / 8;                   // column pairs per thread
    constexpr int NW0 = MT / 32;                 // warps of h = 0
    const int LD = mid_ld(M), LD2 = LD >> 1;
    double* S    = sm;                           // [M][LD]
    double* xs   = sm + (size_t)M * LD;          // [LD]      raw pivot row
    double* pb   = xs + LD;                      // [LD]      p
    double* taus = pb + LD;                      // [LD]
    double* pd   = taus + LD;                    // [MID_TPR][MT] partial products
    double* red  = pd + MID_TPR * MT;            // [2][32]
    const int tid = threadIdx.x, j = tid % MT, h = tid / MT, lane = tid & 31, warp = tid >> 5;
    const size_t b = blockIdx.x;
    const double* A = A_ + b * M * M;
    double* dws = ws.dws + b * M;
    double* ews = ws.ews + b * M;

    // full symmetric copy of the lower triangle: thread (j, h) copies column j of rows h, h+4, ...
    if (j < M)
        for (int r = h; r < M; r += MID_TPR) S[r * LD + j] = (r >= j) ? A[(size_t)r * M + j] : A[(size_t)j * M + r];
    for (int c = tid; c < LD; c += blockDim.x) pb[c] = 0.0;
    __syncthreads();
    double2 a[NP];
    {
        const double2* row2 = reinterpret_cast<const double2*>(S + (size_t)min(j, M - 1) * LD);
#pragma unroll
        for (int k = 0; k < NP; ++k) {
            const int c = 2 * h + 8 * k;
            double2 t = make_double2(0.0, 0.0);
            if (j < M && c < M) { t = row2[h + 4 * k]; if (c + 1 >= M) t.y = 0.0; }
            a[k] = t;
        }
    }
    __syncthreads();                             // S is free: it now collects the reflectors
    const double2* S2 = reinterpret_cast<const double2*>(S);
    double2* xs2 = reinterpret_cast<double2*>(xs);
    auto dump_row = [&]() {                      // the four owners of the next pivot row: raw row -> xs
#pragma unroll
        for (int k = 0; k < NP; ++k)
            if (2 * h + 8 * k < LD) xs2[h + 4 * k] = a[k];
    };
    if (j == M - 1) dump_row();
    for (int i = M - 1; i >= (HEAD ? 64 : 1); --i) {
        __syncthreads();                                                     // B0
        if (h == 0) {
            double part = 0.0;
#pragma unroll
            for (int u = 0; u < MT / 32; ++u) {
                const int c = lane + 32 * u;
                const double x = (c < i - 1) ? xs[c] : 0.0;
                part = fma(x, x, part);
            }
            const double sigma = warp_sum(part);                             // each of the NW0 warps, redundantly
            const double alpha = xs[i - 1];
            double tau = 0.0, scal = 0.0, beta = alpha;                      // sigma == 0: H_i = I (reading G19)
            if (sigma != 0.0) {
                const double nrm2 = fma(alpha, alpha, sigma);
                const double rinv = rsqrt(nrm2);
                beta = -copysign(nrm2 * rinv, alpha);
                tau = fma(fabs(alpha), rinv, 1.0);
                scal = 1.0 / (alpha - beta);
            }
            if (j < LD) S[(size_t)i * LD + j] = (j < i - 1) ? xs[j] * scal : ((j == i - 1) ? 1.0 : 0.0);
            if (j == 0) { dws[i] = xs[i]; ews[i - 1] = beta; taus[i] = tau; }
        }
        __syncthreads();                                                     // B1
        const double tau = taus[i];
        if (tau != 0.0) {                                                    // the same in every thread
            const bool act = (j & ~31) < i;                                  // warp-uniform: a warp of dead rows does nothing
            const double2* v2 = S2 + (size_t)i * LD2 + h;
            if (act) {
                double acc[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
                for (int k = 0; k < NP; ++k) {
                    if (8 * k < i) {
                        const double2 v = v2[4 * k];
                        acc[2 * (k & 1)] = fma(a[k].x, v.x, acc[2 * (k & 1)]);
                        acc[2 * (k & 1) + 1] = fma(a[k].y, v.y, acc[2 * (k & 1) + 1]);
                    }
                }
                pd[h * MT + j] = (acc[0] + acc[1]) + (acc[2] + acc[3]);
            }
            __syncthreads();                                                 // B2
            if (h == 0) {
                double pj = 0.0;
                if (act && j < i) pj = tau * ((pd[j] + pd[MT + j]) + (pd[2 * MT + j] + pd[3 * MT + j]));
                const double vj = (j < i) ? S[(size_t)i * LD + j] : 0.0;
                const double pvw = warp_sum(pj * vj);
                if (j < LD) pb[j] = pj;
                if (lane == 0) red[warp] = pvw;
            }
            __syncthreads();                                                 // B3
            if (act) {
                const double2* p2 = reinterpret_cast<const double2*>(pb) + h;
                double ptv = 0.0;
#pragma unroll
                for (int w = 0; w < NW0; ++w) ptv += red[w];
                const double vj = (j < i) ? S[(size_t)i * LD + j] : 0.0;
                const double pj = (j < i) ? pb[j] : 0.0;
                const double wj = fma(-tau * ptv, vj, pj);                   // p_j - 2 K v_j, K = tau (p.v) / 2
#pragma unroll
                for (int k = 0; k < NP; ++k) {
                    if (8 * k < i) {
                        const double2 v = v2[4 * k], p = p2[4 * k];
                        a[k].x = fma(-vj, p.x, fma(-wj, v.x, a[k].x));
                        a[k].y = fma(-vj, p.y, fma(-wj, v.y, a[k].y));
                    }
                }
            }
        }
        if (j == i - 1) dump_row();
    }
    if constexpr (HEAD) {
        if (tid == 0) ews[M - 1] = 0.0;
        __syncthreads();                                                     // taus, reflector rows complete
        if (j < 64) {                                                        // the trailing block, row j
            double2* row2 = reinterpret_cast<double2*>(blk + b * 4096 + (size_t)j * 64);
#pragma unroll
            for (int k = 0; k < NP; ++k)
                if (2 * h + 8 * k < 64) row2[h + 4 * k] = a[k];
        }
        double* out = ws.refl + b * ws.reflstride + mid_split_fast_doubles();
        const int nrow = M - 64;
        for (int idx = tid; idx < nrow * LD; idx += blockDim.x) out[idx] = S[(size_t)64 * LD + idx];
        for (int c = tid; c < LD; c += blockDim.x) out[(size_t)nrow * LD + c] = (c >= 64 && c <= M - 1) ? taus[c] : 0.0;
        return;
    } else {
    if (tid == 0) { dws[0] = a[0].x; ews[M - 1] = 0.0; }
    __syncthreads();                                                         // taus, reflector rows complete
    mid_formq_rows<MT, MT <= 128>(S, LD, taus, M, V_ + b * M * M);
    }
}

// Q^T of the split reduction: the reflectors of pivots M-1 ... 64 (mid_tridiag_formq_reg<MT, true>) and of
// pivots 63 ... 1 (fast_tridiag<64> / fast_tridiag_tail, RefLayout<64> order) meet in shared memory in the
// layout mid_formq_rows expects (row i = v of H_i: v_c for c < i-1, 1 at i-1, 0 beyond); (d, e) of the
// trailing block, which the register kernels left in d64 / e64 [n][64], go to their places in (dws, ews).
template <int MT>
__global__ void __launch_bounds__(MT * MID_TPR, MT == 96 ? 2 : 1)
mid_formq_split(double* V_, Workspace ws, int M, const double* __restrict__ d64, const double* __restrict__ e64)
{
    extern __shared__ __align__(16) double sm[];
    const int LD = mid_ld(M);
    double* S    = sm;                           // [M][LD]
    double* taus = sm + (size_t)M * LD + 2 * LD; // (same place as in the reduction kernel)
    const int tid = threadIdx.x, nt = blockDim.x;
    const size_t b = blockIdx.x;
    const double* rec = ws.refl + b * ws.reflstride;
    const double* mid = rec + mid_split_fast_doubles();
    const int nrow = M - 64;
    for (int idx = tid; idx < nrow * LD; idx += nt) S[(size_t)64 * LD + idx] = mid[idx];
    for (int c = tid; c < LD; c += nt) taus[c] = (c >= 64) ? mid[(size_t)nrow * LD + c] : ((c >= 1) ? rec[32 * 8 * 9 + c] : 0.0);
    for (int idx = tid; idx < 64 * LD; idx += nt) {
        const int i = idx / LD, c = idx - i * LD;                             // row i = reflector H_i, 1 <= i <= 63
        double v = 0.0;
        if (i >= 1) {
            const int G = (i - 1) >> 3, k = (i - 1) & 7, len = 8 * (G + 1);
            if (c < len) v = rec[32 * G * (G + 1) + k * len + c];
        }
        S[idx] = v;
    }
    if (tid < 64) {
        ws.dws[b * M + tid] = d64[b * 64 + tid];
        if (tid < 63) ws.ews[b * M + tid] = e64[b * 64 + tid];
    }
    __syncthreads();
    mid_formq_rows<MT, MT <= 128>(S, LD, taus, M, V_ + b * M * M);
}

// a5: thread r owns column c0 + r of Q^T (= a row of Q); a rotation (i, i+1) mixes rows i, i+1 of
// Q^T.  The (c, s) of `ms` sweeps are staged per barrier round, double-buffered, straight from the
// log into shared memory with cp.async (no registers: a thread never waits for the log before it
// rotates); inside a round the threads do not depend on each other (each rotates its own column).
// The kernel is chain-latency bound and shared memory (M x 8 B per column) caps the warps per SM,
// so the columns of one matrix may be dealt to the `nsplit` CTAs of a thread-block cluster
// (nsplit = 2 for 96 < M <= 128: three CTAs of 64 columns per SM instead of one of 128).  The
// CTAs of a matrix share nothing but the buffer: V is read as Q^T and written as sorted row-major
// V in place, so every CTA of the cluster must have read its columns before any of them writes
// its rows -- one cluster barrier after the load.
__global__ void __launch_bounds__(160)
mid_apply(double* __restrict__ V_, Workspace ws, int M, int ms, int nsplit, int ncol)
{
    extern __shared__ __align__(16) double sm[];
    const int LD = (ncol + 1) | 1;
    double*   S    = sm;                                                   // [M][LD]  columns c0 ... of Q^T
    double2*  cs   = reinterpret_cast<double2*>(sm + (((size_t)M * LD + 1) & ~(size_t)1));   // [2][ms][M]
    uint32_t* hdr  = reinterpret_cast<uint32_t*>(cs + 2 * ms * M);
    int*      perm = reinterpret_cast<int*>(hdr + ws.swcap);
    const int r = threadIdx.x, nt = blockDim.x;
    const size_t b = blockIdx.x / nsplit;
    const int c0 = (int)(blockIdx.x % nsplit) * ncol;
    const int nc = min(ncol, M - c0);                 // columns of this CTA (<= 0: none)
    if (ws.flags[b]) return;                          // finished by generic_apply (slow path); the whole cluster leaves
    double* V = V_ + b * M * M;
    const int nsw = ws.nsweeps[b];
    const double2* rot = ws.rot + b * ws.logcap;

    for (int s = r; s < nsw; s += nt) hdr[s] = ws.hdr[b * ws.swcap + s];
    if (r < nc)
        for (int k = 0; k < M; ++k) S[k * LD + r] = V[(size_t)k * M + c0 + r];
    for (int k = r; k < M; k += nt) perm[k] = ws.perm[b * M + k];
    if (nsplit > 1) {
        asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    }
    __syncthreads();

    // stage the sweeps [s0, s0 + ms) of the log, which start at log position p0; returns the
    // position after them
    auto stage = [&](int s0, int p0, double2* buf) {
        for (int t = 0; t < ms && s0 + t < nsw; ++t) {
            const uint32_t h = hdr[s0 + t];
            const int n = (int)(h >> 16) - (int)(h & 0xffff);
            for (int k = r; k < n; k += nt) cp_async16(buf + t * M + k, rot + p0 + k);
            p0 += n;
        }
        return p0;
    };
    int pos = stage(0, 0, cs);
    cp_async_wait_all();
    __syncthreads();
    for (int s0 = 0; s0 < nsw; s0 += ms) {
        const double2* cur0 = cs + ((s0 / ms) & 1) * ms * M;
        pos = stage(s0 + ms, pos, cs + (((s0 / ms) + 1) & 1) * ms * M);
        if (r < nc) {
            double* col = S + r;
            for (int t = 0; t < ms && s0 + t < nsw; ++t) {
                const uint32_t h = hdr[s0 + t];
                const int lo = h & 0xffff, m = h >> 16;
                const double2* cur = cur0 + t * M;
                double f = col[m * LD];
                int i = m - 1;
                for (; i - 3 >= lo; i -= 4) {
                    const double2 q0 = cur[m - 1 - i], q1 = cur[m - i], q2 = cur[m + 1 - i], q3 = cur[m + 2 - i];
                    const double z0 = col[i * LD], z1 = col[(i - 1) * LD], z2 = col[(i - 2) * LD], z3 = col[(i - 3) * LD];
                    col[(i + 1) * LD] = fma(q0.y, z0, q0.x * f);  f = fma(-q0.y, f, q0.x * z0);
                    col[i * LD]       = fma(q1.y, z1, q1.x * f);  f = fma(-q1.y, f, q1.x * z1);
                    col[(i - 1) * LD] = fma(q2.y, z2, q2.x * f);  f = fma(-q2.y, f, q2.x * z2);
                    col[(i - 2) * LD] = fma(q3.y, z3, q3.x * f);  f = fma(-q3.y, f, q3.x * z3);
                }
                for (; i >= lo; --i) {
                    const double2 q = cur[m - 1 - i];
                    const double zi = col[i * LD];
                    col[(i + 1) * LD] = fma(q.y, zi, q.x * f);
                    f = fma(-q.y, f, q.x * zi);
                }
                col[lo * LD] = f;
            }
        }
        cp_async_wait_all();
        __syncthreads();
    }

    // V[c0 + row][k] = Qt'[perm[k]][c0 + row]: one warp per output row, lanes over the sorted columns
    const int lane = r & 31, warp = r >> 5, nw = nt >> 5;
    for (int row = warp; row < nc; row += nw)
        for (int k = lane; k < M; k += 32) V[(size_t)(c0 + row) * M + k] = S[perm[k] * LD + row];
}

}  // namespace letkf

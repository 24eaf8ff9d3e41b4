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
static inline size_t mid_apply_smem(int M, int swcap, int ms)
{
    return sizeof(double) * ((size_t)M * (M + 1) + 4 * (size_t)ms * (size_t)M) + sizeof(uint32_t) * (size_t)swcap + sizeof(int) * (size_t)M + 32;
}
// sweeps staged per barrier round of mid_apply: as many (<= 4) as shared memory holds beside the matrix
static inline int mid_apply_round(int M, int swcap)
{
    int ms = 4;
    while (ms > 1 && mid_apply_smem(M, swcap, ms) > 226 * 1024) ms >>= 1;
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

// MID_TPR threads per row: thread (j, h) = (tid % RP, tid / RP), RP = ceil32(M), owns the column
// pairs p = h, h + TPR, ... of row j (16-byte accesses); the partial products of a row meet in
// shared memory.  vs / wsm are kept zero at index i (the first dead column) so that a pair that
// straddles the active range contributes nothing.
__global__ void __launch_bounds__(160 * MID_TPR)
mid_tridiag_formq(const double* __restrict__ A_, double* V_, Workspace ws, int M)
{
    extern __shared__ __align__(16) double sm[];
    const int LD = mid_ld(M);
    const int RP = blockDim.x / MID_TPR;
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
        if (h == 1 && j == 0) S[i * LD + i] = 0.0;                 // update touches it); (pair overhang)
        __syncthreads();
    }
    if (tid == 0) { dws[0] = S[0]; ews[M - 1] = 0.0; }

    // Q^T = H_1 H_2 ... H_{M-1}, grown in place: B_i = diag(B_{i-1}, 1) H_i on the leading i x i
    for (int i = 1; i <= M - 1; ++i) {
        if (h == 0) {
            if (j < i) vs[j] = S[i * LD + j];
            if (j == i) vs[j] = 0.0;
        }
        const double tau = taus[i];
        __syncthreads();                                           // reflector copied before row i-1 ... are cleared
        if (h == 0 && j < i - 1) { S[(i - 1) * LD + j] = 0.0; S[j * LD + (i - 1)] = 0.0; }
        if (h == 1 && j == 0) S[(i - 1) * LD + (i - 1)] = 1.0;
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
            if (j < i) {
                double acc = 0.0;
#pragma unroll
                for (int hh = 0; hh < MID_TPR; ++hh) acc += pd[hh * RP + j];
                acc *= -tau;
#pragma unroll 4
                for (int p = h; p < npair; p += MID_TPR) {
                    double2 r = row2w[p];
                    const double2 v = v2[p];
                    r.x = fma(acc, v.x, r.x);
                    r.y = fma(acc, v.y, r.y);
                    row2w[p] = r;
                }
            }
        }
        __syncthreads();
    }
    if (h == 0 && j < M - 1) { S[(M - 1) * LD + j] = 0.0; S[j * LD + (M - 1)] = 0.0; }
    __syncthreads();
    if (tid == 0) S[(M - 1) * LD + (M - 1)] = 1.0;
    __syncthreads();
    if (j < M) {
        double* Qt = V_ + b * M * M;
        for (int r = h; r < M; r += MID_TPR) Qt[(size_t)r * M + j] = S[r * LD + j];
    }
}

// a5: thread r owns column r of Q^T (= row r of Q); a rotation (i, i+1) mixes rows i, i+1 of Q^T.
// The (c, s) of `ms` sweeps are staged per barrier round, double-buffered, straight from the log
// into shared memory with cp.async (no registers: a thread never waits for the log before it
// rotates); inside a round the threads do not depend on each other (each rotates its own column).
__global__ void __launch_bounds__(160)
mid_apply(double* __restrict__ V_, Workspace ws, int M, int ms)
{
    extern __shared__ __align__(16) double sm[];
    const int LD = M + 1;
    double*   S    = sm;                                                   // [M][LD]  Q^T
    double2*  cs   = reinterpret_cast<double2*>(sm + (((size_t)M * LD + 1) & ~(size_t)1));   // [2][ms][M]
    uint32_t* hdr  = reinterpret_cast<uint32_t*>(cs + 2 * ms * M);
    int*      perm = reinterpret_cast<int*>(hdr + ws.swcap);
    const int r = threadIdx.x, nt = blockDim.x;
    const size_t b = blockIdx.x;
    if (ws.flags[b]) return;                          // finished by generic_apply (slow path)
    double* V = V_ + b * M * M;
    const int nsw = ws.nsweeps[b];
    const double2* rot = ws.rot + b * ws.logcap;

    for (int s = r; s < nsw; s += nt) hdr[s] = ws.hdr[b * ws.swcap + s];
    if (r < M) {
        for (int k = 0; k < M; ++k) S[k * LD + r] = V[(size_t)k * M + r];
        perm[r] = ws.perm[b * M + r];
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
        if (r < M) {
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

    // V[row][k] = Qt'[perm[k]][row]: one warp per output row, lanes over the sorted columns
    const int lane = r & 31, warp = r >> 5, nw = nt >> 5;
    for (int row = warp; row < M; row += nw)
        for (int k = lane; k < M; k += 32) V[(size_t)row * M + k] = S[perm[k] * LD + row];
}

}  // namespace letkf

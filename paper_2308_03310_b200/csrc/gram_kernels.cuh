// gram_kernels.cuh -- a1 + a2 for the orders above the register kernels (M > 64), on the FP64 tensor cores.
//
//   A[m][n] = ((M-1)/rho) delta_mn + sum_j r_j Yb[j][m] Yb[j][n]     (Eq.17)
//   g[m]    = sum_j Yb[j][m] r_j d_j                                  (right factor of Eq.14)
//
// The Gram matrix is the one dense contraction of the path; for M <= 64 it runs as
// mma.sync.m8n8k4.f64 inside the reduction kernel (fast_kernels.cuh), above that generic_gram formed it with a
// 4 x 4 register tile per thread from global memory.  Here: one CTA of 8 warps per grid point, the observations
// Yb[j0 .. j0+pj)[0 .. M) staged once in shared memory (row stride = 4 mod 16 doubles: both operand fragments
// are "lane l: row 4 kk + l mod 4, column base + l div 4", conflict-free per half warp), a warp owns 32 x 32
// blocks of the lower triangle (16 accumulator tiles of 8 x 8) and walks the observations four at a time:
// eight shared-memory loads feed sixteen DMMA (4096 FMA).  Only the blocks on and below the diagonal are formed
// (every reduction kernel reads the lower triangle).  p larger than shared memory holds: chunks, accumulated
// in the output.
#pragma once
#include "common.cuh"
#include "ns_kernel.cuh"

namespace letkf {

constexpr int GRAM_NT = 256;
constexpr size_t GRAM_SMEM_CAP = 224 * 1024;

static inline int gram_ld(int M) { return (M + 31) / 32 * 32 + 4; }     // whole 32-column blocks, = 4 mod 16
// observations staged per chunk (a multiple of 4)
static inline int gram_chunk(int M, int p)
{
    const int cap = (int)((GRAM_SMEM_CAP / sizeof(double)) / (size_t)(gram_ld(M) + 2)) & ~3;
    const int need = (p + 3) & ~3;
    return need < cap ? (need > 4 ? need : 4) : cap;
}
static inline size_t gram_smem(int M, int p) { return sizeof(double) * (size_t)gram_chunk(M, p) * (gram_ld(M) + 2); }

// Yb: [batch][p][M], d, r: [batch][p]; Aout: [batch][M][M] (lower triangle and the rest of the diagonal blocks
// written), gout: [batch][M].  PJ = gram_chunk(M, p).
__global__ void __launch_bounds__(GRAM_NT)
big_gram(const double* __restrict__ Yb_, const double* __restrict__ d_, const double* __restrict__ r_,
         int M, int p, int PJ, double shift, double* __restrict__ Aout_, double* __restrict__ gout_)
{
    extern __shared__ __align__(16) double gr_sm[];
    const int LD = (M + 31) / 32 * 32 + 4;
    double* Ys = gr_sm;                        // [PJ][LD]
    double* rs = Ys + (size_t)PJ * LD;         // [PJ] r_j
    double* rd = rs + PJ;                      // [PJ] r_j d_j
    const size_t b = blockIdx.x;
    const double* Yb = Yb_ + b * (size_t)p * M;
    const double* dv = d_ + b * (size_t)p;
    const double* rv = r_ + b * (size_t)p;
    double* Aout = Aout_ + b * (size_t)M * M;
    double* gout = gout_ + b * M;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int NB = (M + 31) >> 5, nblocks = NB * (NB + 1) / 2;

    for (int j0 = 0, first = 1; first || j0 < p; j0 += PJ, first = 0) {
        const int pj = min(PJ, p - j0);                         // observations of this chunk (0 when p = 0)
        const int pj4 = (pj + 3) & ~3;
        __syncthreads();                                        // (the previous chunk is done with the tile)
        for (int idx = tid; idx < pj4 * LD; idx += GRAM_NT) {
            const int j = idx / LD, c = idx - j * LD;
            Ys[idx] = (j < pj && c < M) ? Yb[(size_t)(j0 + j) * M + c] : 0.0;
        }
        for (int j = tid; j < pj4; j += GRAM_NT) {
            const double rj = (j < pj) ? rv[j0 + j] : 0.0;
            rs[j] = rj;
            rd[j] = (j < pj) ? rj * dv[j0 + j] : 0.0;
        }
        __syncthreads();
        for (int m = tid; m < M; m += GRAM_NT) {                // a2
            double acc = first ? 0.0 : gout[m];
            for (int j = 0; j < pj; ++j) acc = fma(Ys[(size_t)j * LD + m], rd[j], acc);
            gout[m] = acc;
        }
        for (int t = warp; t < nblocks; t += GRAM_NT / 32) {    // a1: block (bm, bn), bn <= bm
            int bm = 0, rem = t;
            while (rem > bm) { rem -= bm + 1; ++bm; }
            const int bn = rem;
            double acc[4][4][2];
#pragma unroll
            for (int rt = 0; rt < 4; ++rt)
#pragma unroll
                for (int ct = 0; ct < 4; ++ct) { acc[rt][ct][0] = 0.0; acc[rt][ct][1] = 0.0; }
            const double* ya = Ys + (size_t)(lane & 3) * LD + 32 * bm + (lane >> 2);   // (the tile is zero beyond column M)
            const double* yb = Ys + (size_t)(lane & 3) * LD + 32 * bn + (lane >> 2);
            for (int kk = 0; kk < pj4; kk += 4) {
                const double rj = rs[kk + (lane & 3)];
                double a[4], bq[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    a[u] = rj * ya[(size_t)kk * LD + 8 * u];
                    bq[u] = yb[(size_t)kk * LD + 8 * u];
                }
#pragma unroll
                for (int rt = 0; rt < 4; ++rt)
#pragma unroll
                    for (int ct = 0; ct < 4; ++ct) dmma884(acc[rt][ct], a[rt], bq[ct]);
            }
#pragma unroll
            for (int rt = 0; rt < 4; ++rt)
#pragma unroll
                for (int ct = 0; ct < 4; ++ct) {
                    const int m = 32 * bm + 8 * rt + (lane >> 2);
                    const int n = 32 * bn + 8 * ct + 2 * (lane & 3);
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        if (m < M && n + e < M) {
                            double* out = Aout + (size_t)m * M + n + e;
                            double val = acc[rt][ct][e];
                            if (first) { if (m == n + e) val += shift; }
                            else val += *out;
                            *out = val;
                        }
                    }
                }
        }
    }
}

}  // namespace letkf

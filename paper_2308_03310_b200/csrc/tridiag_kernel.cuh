// tridiag_kernel.cuh -- steps a3 (+ a1/a2 when fused) and the explicit Q for M <= 64:
// Householder tridiagonalisation with the matrix REGISTER-RESIDENT (PAPER.md:183 names the
// algorithm; the mapping is ours).
//
//   thread j owns row j of the symmetric work matrix, a[0..MT-1], in registers;
//   the reduction runs from the last row up: pivot i = M-1 ... 1, reflector H_i acts on indices
//   0..i-1, so T = Q^T A Q with Q = H_{M-1} ... H_1;
//   afterwards thread r forms column r of Q (q <- H_i q for i = r+1 ... M-1: no communication).
//
// Register arrays need compile-time indices, so the pivot loop is cut into GROUPS of 8 pivots
// (template parameter G: i in 8G+1 .. 8G+8); inside a group every vector operation covers the
// same 8(G+1) columns and is straight-line code -- no jump tables, and the compiler is free to
// software-pipeline the shared-memory broadcasts.  Vectors in shared memory are kept ZERO beyond
// the active length so the (at most 7-column) overhang contributes nothing.
//
// Shared memory is addressed through 32-bit shared-window addresses with ld.shared/st.shared:
// with generic pointers ptxas re-derived the window base (S2UR SR_CgaCtaId + ULEA, ~40 cycles)
// in front of every block of loads (profiles/r01_ncu_fast_v1.md).
#pragma once
#include "common.cuh"

namespace letkf {

__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ double2 lds128(uint32_t a)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ double lds64(uint32_t a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts64(uint32_t a, double v)
{
    asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory");
}
__device__ __forceinline__ void sts128(uint32_t a, double2 v)
{
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(v.x), "d"(v.y) : "memory");
}

template <int MT> struct FastCfg {
    static constexpr int NT = (MT + 31) / 32 * 32;      // threads per matrix = threads per CTA
    static constexpr int NW = NT / 32;
    static constexpr int LDT = MT + 1;                  // padded tile stride (doubles)
    static constexpr int NG = MT / 8;                   // pivot groups
    // byte offsets into the dynamic shared memory of fast_tridiag_formq
    static constexpr uint32_t OFF_TILE = 0;                               // A staging, later R[i][c]
    static constexpr uint32_t OFF_VS   = 8u * MT * (MT + 1);              // v            [MT]
    static constexpr uint32_t OFF_VP   = OFF_VS + 8u * MT;                // (v, p) pairs [MT]
    static constexpr uint32_t OFF_TAU  = OFF_VP + 16u * MT;               // tau          [MT]
    static constexpr uint32_t OFF_RED  = OFF_TAU + 8u * MT;               // scratch      [8]
    static constexpr uint32_t SMEM     = OFF_RED + 64u;
};

// Barrier over the first NP warps of the CTA (named barrier 1; __syncwarp when NP == 1).
template <int NP>
__device__ __forceinline__ void part_barrier()
{
    if constexpr (NP <= 1) __syncwarp();
    else asm volatile("bar.sync 1, %0;" ::"n"(NP * 32) : "memory");
}

// sum_{c < 8 NB} a[c] * vec[c]
template <int MT, int NB>
__device__ __forceinline__ double dot_blocks(const double (&a)[MT], uint32_t vec)
{
    double s[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) s[k] = 0.0;
#pragma unroll
    for (int g = 0; g < NB; ++g)
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            const double2 t = lds128(vec + 8u * (8 * g + 2 * h));
            s[2 * h]     = fma(a[8 * g + 2 * h],     t.x, s[2 * h]);
            s[2 * h + 1] = fma(a[8 * g + 2 * h + 1], t.y, s[2 * h + 1]);
        }
    return ((s[0] + s[1]) + (s[2] + s[3])) + ((s[4] + s[5]) + (s[6] + s[7]));
}

// a[c] -= alpha * vec[c],  c < 8 NB
template <int MT, int NB>
__device__ __forceinline__ void axpy_blocks(double (&a)[MT], uint32_t vec, double alpha)
{
    const double na = -alpha;
#pragma unroll
    for (int g = 0; g < NB; ++g)
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            const double2 t = lds128(vec + 8u * (8 * g + 2 * h));
            a[8 * g + 2 * h]     = fma(na, t.x, a[8 * g + 2 * h]);
            a[8 * g + 2 * h + 1] = fma(na, t.y, a[8 * g + 2 * h + 1]);
        }
}

// a[c] -= vj * p[c] + wj * v[c],  c < 8 NB;  vp[c] = (v_c, p_c)
template <int MT, int NB>
__device__ __forceinline__ void rank2_blocks(double (&a)[MT], uint32_t vp, double vj, double wj)
{
    const double nv = -vj, nw = -wj;
#pragma unroll
    for (int c = 0; c < 8 * NB; ++c) {
        const double2 t = lds128(vp + 16u * c);
        a[c] = fma(nv, t.y, fma(nw, t.x, a[c]));
    }
}

// a[i] for i in 8G+1 .. 8G+8 (warp-uniform i): predicated moves, no jump table
template <int MT, int G>
__device__ __forceinline__ double pick_group(const double (&a)[MT], int i)
{
    double x = 0.0;
#pragma unroll
    for (int k = 1; k <= 8; ++k)
        if constexpr (8 * G + k < MT) {
            if (i == 8 * G + k) x = a[8 * G + k];
        }
    return x;
}

// a[i] for an arbitrary (per-thread) index: used once per thread, for the diagonal
template <int MT>
__device__ __forceinline__ double pick_any(const double (&a)[MT], int i)
{
    double x = 0.0;
#pragma unroll
    for (int c = 0; c < MT; ++c)
        if (i == c) x = a[c];
    return x;
}

// One group of pivots i = min(M-1, 8G+8) ... 8G+1 of the reduction.  Called by the warps that
// still own active rows (rows j < i): warps 0 .. NP-1 with NP = G/4 + 1.
template <int MT, int G>
__device__ __forceinline__ void tridiag_group(double (&a)[MT], int M, uint32_t sb, double* __restrict__ ews)
{
    using C = FastCfg<MT>;
    constexpr int NP = (G / 4 + 1 < C::NW) ? G / 4 + 1 : C::NW;
    constexpr int NB = G + 1;
    const int j = threadIdx.x, lane = j & 31, warp = j >> 5;
    const uint32_t red = sb + C::OFF_RED, vs = sb + C::OFF_VS, vp = sb + C::OFF_VP;
    const int ihi = (M - 1 < 8 * G + 8) ? M - 1 : 8 * G + 8;
    for (int i = ihi; i >= 8 * G + 1; --i) {
        const double x = pick_group<MT, G>(a, i);          // x_j = A[j][i]
        if (j == i - 1) sts64(red + 32, x);                // alpha
        double part = (j < i - 1) ? x * x : 0.0;
        part = warp_sum(part);
        if (lane == 0) sts64(red + 8u * warp, part);
        part_barrier<NP>();
        double sigma = lds64(red);
        if constexpr (NP > 1) sigma += lds64(red + 8);
        const double alpha = lds64(red + 32);
        double tau, scal, beta;
        if (sigma == 0.0) { tau = 0.0; beta = alpha; scal = 0.0; }       // reading G19: H_i = I
        else {
            const double nrm2 = fma(alpha, alpha, sigma);
            const double rinv = rsqrt(nrm2);
            const double nrm = nrm2 * rinv;
            beta = -copysign(nrm, alpha);
            tau = fma(fabs(alpha), rinv, 1.0);                            // (beta - alpha)/beta
            scal = 1.0 / (alpha - beta);
        }
        const double vj = (j < i - 1) ? x * scal : ((j == i - 1) ? 1.0 : 0.0);
        if (j < MT) {
            sts64(vs + 8u * j, vj);
            sts64(sb + C::OFF_TILE + 8u * (i * MT + j), vj);             // reflector R[i][j]
        }
        if (j == 0) { ews[i - 1] = beta; sts64(sb + C::OFF_TAU + 8u * i, tau); }
        part_barrier<NP>();
        if (tau != 0.0) {
            double pj = tau * dot_blocks<MT, NB>(a, vs);                  // p = tau A v
            if (j >= i) pj = 0.0;
            const double pv = warp_sum(pj * vj);
            if (lane == 0) sts64(red + 16 + 8u * warp, pv);
            if (j < MT) sts128(vp + 16u * j, make_double2(vj, pj));
            part_barrier<NP>();
            double ptv = lds64(red + 16);
            if constexpr (NP > 1) ptv += lds64(red + 24);
            // A -= v w^T + w v^T, w = p - (tau/2)(p.v) v, on the broadcast pairs (v_c, p_c):
            //   a_jc -= v_j p_c + (p_j - tau (p.v) v_j) v_c
            const double wj = pj - (tau * ptv) * vj;
            if (j < i) rank2_blocks<MT, NB>(a, vp, vj, wj);
        }
    }
}

// groups G = GTOP ... 0, each run by the warps that still take part
template <int MT, int G>
__device__ __forceinline__ void tridiag_groups(double (&a)[MT], int M, uint32_t sb, double* __restrict__ ews)
{
    using C = FastCfg<MT>;
    constexpr int NP = (G / 4 + 1 < C::NW) ? G / 4 + 1 : C::NW;
    if ((int)(threadIdx.x >> 5) >= NP) return;            // this warp's rows are all reduced
    if (8 * G + 1 <= M - 1) tridiag_group<MT, G>(a, M, sb, ews);
    if constexpr (G > 0) tridiag_groups<MT, G - 1>(a, M, sb, ews);
}

// q <- H_i q for i = 8G+1 ... min(M-1, 8G+8): thread-local, reflectors read from shared memory
template <int MT, int G>
__device__ __forceinline__ void formq_groups(double (&q)[MT], int M, uint32_t sb, int gfirst)
{
    using C = FastCfg<MT>;
    constexpr int NB = G + 1;
    if (G >= gfirst) {
        const int ihi = (M - 1 < 8 * G + 8) ? M - 1 : 8 * G + 8;
        for (int i = 8 * G + 1; i <= ihi; ++i) {
            const double tau = lds64(sb + C::OFF_TAU + 8u * i);
            if (tau == 0.0) continue;
            const uint32_t v = sb + C::OFF_TILE + 8u * (i * MT);
            const double s = tau * dot_blocks<MT, NB>(q, v);
            axpy_blocks<MT, NB>(q, v, s);
        }
    }
    if constexpr (G + 1 < C::NG) formq_groups<MT, G + 1>(q, M, sb, gfirst);
}

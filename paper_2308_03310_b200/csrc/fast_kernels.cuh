// fast_kernels.cuh -- register-resident path for M <= 64 (the paper's sizes, Table I,
// and the headline M = 64).
//
// Design: a matrix lives in the REGISTERS of MT threads, one row (or one
// column) per thread, for its whole life inside a kernel.  An SM issues 64 fp64 FMAs per clock but
// shared memory delivers only 16 doubles per clock, so BLAS-2 work fed from shared memory cannot
// pass 25% of the fp64 peak; here shared memory only carries the broadcast vectors (one LDS.128
// feeds two FMAs in every lane).  Register arrays need compile-time indices: the reduction runs in
// groups of 8 pivots with statically shaped 8-column block loops (pivot_group<G>), the rotation
// replay in blocks of 4 rotations entered through a switch with fall-through cases (apply_sweep).
//
//   fast_tridiag<MT>   a3 (+ a1, a2)   : thread j = row j of A; leaves (d, e) and the reflectors
//   ql_log_kernel      a4              : ql_kernel.cuh, one thread per matrix, rotations logged
//   fast_apply<MT>     a5 (+ a6-a9)    : thread r = row r of Z (from I): replays the log; the matrix
//                                        is turned through shared memory and thread k applies the
//                                        reflectors to eigenvector k: V = H_{M-1} ... H_1 Z
// Q is never formed and the matrix crosses HBM once in (A) and once out (V).
#pragma once
#include "common.cuh"

namespace letkf {

// X(31) X(30) ... X(0)
#define LETKF_REP32_DESC(X) \
    X(31) X(30) X(29) X(28) X(27) X(26) X(25) X(24) X(23) X(22) X(21) X(20) X(19) X(18) X(17) X(16) \
    X(15) X(14) X(13) X(12) X(11) X(10) X(9) X(8) X(7) X(6) X(5) X(4) X(3) X(2) X(1) X(0)
#define LETKF_REP64_DESC(X) \
    X(63) X(62) X(61) X(60) X(59) X(58) X(57) X(56) X(55) X(54) X(53) X(52) X(51) X(50) X(49) X(48) \
    X(47) X(46) X(45) X(44) X(43) X(42) X(41) X(40) X(39) X(38) X(37) X(36) X(35) X(34) X(33) X(32) \
    X(31) X(30) X(29) X(28) X(27) X(26) X(25) X(24) X(23) X(22) X(21) X(20) X(19) X(18) X(17) X(16) \
    X(15) X(14) X(13) X(12) X(11) X(10) X(9) X(8) X(7) X(6) X(5) X(4) X(3) X(2) X(1) X(0)

// ---- the real type of the register path: double (everything), or float for the reduction, the
// replay and the back-transform of letkf_syev_batched_f32
template <typename R> struct Blk8;        // 8 consecutive entries of a broadcast vector in shared memory
template <> struct Blk8<double> {
    double2 t0, t1, t2, t3;               // four LDS.128, each feeds two FMAs in every lane
    __device__ __forceinline__ Blk8(const double* vec, int g)
    {
        const double2* v2 = reinterpret_cast<const double2*>(vec);
        t0 = v2[4 * g]; t1 = v2[4 * g + 1]; t2 = v2[4 * g + 2]; t3 = v2[4 * g + 3];
    }
    __device__ __forceinline__ double v0() const { return t0.x; }
    __device__ __forceinline__ double v1() const { return t0.y; }
    __device__ __forceinline__ double v2() const { return t1.x; }
    __device__ __forceinline__ double v3() const { return t1.y; }
    __device__ __forceinline__ double v4() const { return t2.x; }
    __device__ __forceinline__ double v5() const { return t2.y; }
    __device__ __forceinline__ double v6() const { return t3.x; }
    __device__ __forceinline__ double v7() const { return t3.y; }
};
template <> struct Blk8<float> {
    float4 t0, t1;                        // two LDS.128, each feeds four FMAs
    __device__ __forceinline__ Blk8(const float* vec, int g)
    {
        const float4* v4 = reinterpret_cast<const float4*>(vec);
        t0 = v4[2 * g]; t1 = v4[2 * g + 1];
    }
    __device__ __forceinline__ float v0() const { return t0.x; }
    __device__ __forceinline__ float v1() const { return t0.y; }
    __device__ __forceinline__ float v2() const { return t0.z; }
    __device__ __forceinline__ float v3() const { return t0.w; }
    __device__ __forceinline__ float v4() const { return t1.x; }
    __device__ __forceinline__ float v5() const { return t1.y; }
    __device__ __forceinline__ float v6() const { return t1.z; }
    __device__ __forceinline__ float v7() const { return t1.w; }
};
__device__ __forceinline__ double rsq(double x) { return rsqrt(x); }
__device__ __forceinline__ float rsq(float x) { return rsqrtf(x); }

// register-array read with a run-time index (jump table; indices stay compile-time constants)
template <int MT, typename R>
__device__ __forceinline__ R pick(const R (&a)[MT], int i)
{
    R x = R(0);
    switch (i) {
#define LETKF_PICK(c) case c: if constexpr (c < MT) x = a[c]; break;
        LETKF_REP64_DESC(LETKF_PICK)
#undef LETKF_PICK
    }
    return x;
}

// ---- statically shaped BLAS-1 pieces of the reduction (pivot group G: columns 0 .. 8G+7) -----
// Inside a group of 8 pivots the active column range rounds up to the same 8-column block, so
// every loop below has compile-time bounds: straight-line code, no jump table, and the compiler is
// free to hoist the shared-memory loads of a whole pass.

// sum_{c < 8(G+1)} a[c] * vec[c]
template <int MT, int G, bool FENCED = false, typename R>
__device__ __forceinline__ R dot_blocks(const R (&a)[MT], const R* vec)
{
    R s0 = R(0), s1 = R(0), s2 = R(0), s3 = R(0), s4 = R(0), s5 = R(0), s6 = R(0), s7 = R(0);
#pragma unroll
    for (int g = G; g >= 0; --g) {
        const Blk8<R> t(vec, g);
        s0 = fma(a[8 * g],     t.v0(), s0); s1 = fma(a[8 * g + 1], t.v1(), s1);
        s2 = fma(a[8 * g + 2], t.v2(), s2); s3 = fma(a[8 * g + 3], t.v3(), s3);
        s4 = fma(a[8 * g + 4], t.v4(), s4); s5 = fma(a[8 * g + 5], t.v5(), s5);
        s6 = fma(a[8 * g + 6], t.v6(), s6); s7 = fma(a[8 * g + 7], t.v7(), s7);
        if constexpr (FENCED) __syncwarp();     // ptxas does not move shared loads across it
    }
    return ((s0 + s1) + (s2 + s3)) + ((s4 + s5) + (s6 + s7));
}

// a[c] -= alpha * vec[c] for the 8 columns of block g
template <int MT, typename R>
__device__ __forceinline__ void axpy_block(R (&a)[MT], const R* vec, R nalpha, int g)
{
    const Blk8<R> t(vec, g);
    a[8 * g]     = fma(nalpha, t.v0(), a[8 * g]);     a[8 * g + 1] = fma(nalpha, t.v1(), a[8 * g + 1]);
    a[8 * g + 2] = fma(nalpha, t.v2(), a[8 * g + 2]); a[8 * g + 3] = fma(nalpha, t.v3(), a[8 * g + 3]);
    a[8 * g + 4] = fma(nalpha, t.v4(), a[8 * g + 4]); a[8 * g + 5] = fma(nalpha, t.v5(), a[8 * g + 5]);
    a[8 * g + 6] = fma(nalpha, t.v6(), a[8 * g + 6]); a[8 * g + 7] = fma(nalpha, t.v7(), a[8 * g + 7]);
}

// a[8G + k], k = 0..7 at run time (select chain; the block is compile-time)
template <int MT, int G, typename R>
__device__ __forceinline__ R block_pick(const R (&a)[MT], int k)
{
    R x = a[8 * G];
#pragma unroll
    for (int t = 1; t < 8; ++t) x = (k == t) ? a[8 * G + t] : x;
    return x;
}

#ifndef LETKF_AP48
#define LETKF_AP48 6      // CTAs per SM of fast_apply<48>: 7 (144 registers) spills 416 B and measured 2.06 ms at config 5, 6 (168) 1.70 ms
#endif
#ifndef LETKF_TRI_REGS64
#define LETKF_TRI_REGS64 168
#endif
#ifndef LETKF_TRI_REGS64_HEAD
#define LETKF_TRI_REGS64_HEAD 200     // the head kernel of the split reduction: 5 CTAs per SM without spills (1.07 ms)
#endif                                // beats 6 with 364 B of spills inside the pivot loop (1.22 ms)
template <int MT> struct FastCfg {
    static constexpr int NT = (MT + 31) / 32 * 32;      // threads per matrix = threads per CTA
    static constexpr int NW = NT / 32;
    static constexpr int LDT = MT + 1;                  // padded tile stride (doubles)
};

// Sum over the CTA of one double per thread, MT <= 64: warp shuffle + one shared slot per warp.
// Costs one __syncthreads; `slot` is a 2-double scratch that must not be reused before the next
// barrier of the caller.
template <int NW>
__device__ __forceinline__ double cta_sum(double v, double* slot)
{
    v = warp_sum(v);
    if constexpr (NW == 1) return v;
    if ((threadIdx.x & 31) == 0) slot[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < NW; ++w) t += slot[w];
    return t;
}

// Barrier over the first `nwarps` warps of the CTA (named barrier 1; __syncwarp when one warp).
__device__ __forceinline__ void part_barrier(int nwarps)
{
    if (nwarps <= 1) __syncwarp();
    else asm volatile("bar.sync 1, %0;" ::"r"(nwarps * 32) : "memory");
}

// Coalesced copy of rows [r0, r0+nr) of a row-major M x M matrix into the padded shared tile
// (tile row = matrix row - r0).  Thread t owns column t: no index arithmetic beyond one add per
// row (a flat index split by a run-time M cost an integer division per element and 17% of the
// tridiagonalisation kernel, profiles/r01b), 8 loads in flight per thread.
template <int MT, typename R>
__device__ __forceinline__ void load_rows(R* tile, const R* __restrict__ G, int M, int r0, int nr)
{
    using C = FastCfg<MT>;
    const int t = threadIdx.x;
    if (t >= M) return;
    const R* src = G + (size_t)r0 * M + t;
    R* dst = tile + t;
    int r = 0;
    for (; r + 8 <= nr; r += 8) {
        R tmp[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) tmp[u] = src[(size_t)(r + u) * M];
#pragma unroll
        for (int u = 0; u < 8; ++u) dst[(r + u) * C::LDT] = tmp[u];
    }
    for (; r < nr; ++r) dst[r * C::LDT] = src[(size_t)r * M];
}

// Reflector storage: H_i (i-1 in [8G, 8G+7]) is only ever read over the 8(G+1) columns of its
// pivot group, so its row is that long: group G starts at 32 G (G+1) doubles.
template <int MT> struct RefLayout {
    static constexpr int GMAX = (MT - 2) / 8;
    static constexpr int TOTAL = 32 * (GMAX + 1) * (GMAX + 2);
    static constexpr int HT = MT < 32 ? MT : 32;                 // rows of A staged per pass
    static constexpr int STAGE = HT * (MT + 1);
    static constexpr int REGION = ((TOTAL > STAGE ? TOTAL : STAGE) + 1) & ~1;   // doubles
    __device__ static constexpr int base(int G) { return 32 * G * (G + 1); }
    __device__ static constexpr int len(int G) { return 8 * (G + 1); }
};

// Back-transform: reflectors i = 8G+1 ... 8G+8 applied to the column q held by this thread.  The
// __syncwarp() after every 8-column block is a scheduling fence: ptxas does not move shared-memory
// loads across it, and without it the loads of a whole pass are hoisted and the matrix spills.
template <int MT, int G, typename R>
__device__ __forceinline__ void q_group(R (&q)[MT], const R* Rf, const R* taus, int M)
{
#pragma unroll 1
    for (int i = 8 * G + 1; i <= 8 * G + 8 && i <= M - 1; ++i) {
        const R tau1 = taus[i];
        if (tau1 == R(0)) continue;
        const R* v1 = Rf + RefLayout<MT>::base(G) + (i - 1 - 8 * G) * RefLayout<MT>::len(G);
        const R ns1 = -tau1 * dot_blocks<MT, G, true>(q, v1);
#pragma unroll
        for (int g = G; g >= 0; --g) { axpy_block<MT>(q, v1, ns1, g); __syncwarp(); }
    }
}

template <int MT, int G, int GMAX, typename R>
__device__ __forceinline__ void q_groups_up(R (&q)[MT], const R* Rf, const R* taus, int M, int gstart)
{
    if (G >= gstart) q_group<MT, G>(q, Rf, taus, M);
    if constexpr (G < GMAX) q_groups_up<MT, G + 1, GMAX>(q, Rf, taus, M, gstart);
}

// Dynamic shared memory of fast_tridiag_formq<MT>:
//   region[RefLayout::REGION]  staging of A, 32 padded rows per pass, later the reflectors
//   xs[NT] raw pivot column;  vbuf[NT] v;  pbuf[NT] p;  pv[NT] p_j v_j;  taus[NT];  red[8]
template <int MT, typename R = double> constexpr size_t fast_tridiag_smem()
{
    return sizeof(R) * ((size_t)RefLayout<MT>::REGION + 5 * FastCfg<MT>::NT + 8);
}

template <typename R> struct TriShared {
    R* Rf;      // reflector storage, RefLayout<MT>
    R* xs;      // x_c = A[c][i] for c < i-1, zero from i-1 on
    R* vbuf;    // v_c (v_{i-1} = 1, zero from i on)
    R* pbuf;    // p_c = tau (A v)_c, zero from i on
    R* pv;      // p_c v_c
    R* taus;
    R* red;     // [0..1] per-warp partial of sigma, [4] alpha
};

// Pivots i = min(8G+8, M-1) ... 8G+1 of the Householder reduction (H_i acts on indices 0..i-1, the
// active columns all lie in blocks 0..G).  Two barriers per pivot:
//   B1  the raw pivot column x and the partial sums of sigma are visible (both were produced by
//       the look-ahead at the end of the previous pivot)
//       -> every thread forms the scalars (tau, beta, 1/(alpha-beta)) redundantly WHILE it runs the
//          raw product sum_c a_jc x_c; then p_j, v_j
//   B2  v, p and the products p_c v_c are visible
//       -> pass A  a_jc -= v_j p_c  overlaps the shuffle tree of p.v
//       -> pass B  a_jc -= (p_j - tau (p.v) v_j) v_c, top block first: column i-1 is then final, it
//          is the next pivot's x, whose norm tree overlaps the rest of pass B.
// Entered and left with B1 done (by the NP warps that hold rows < 8G+8).
// `j` is the row this thread holds (threadIdx.x, or the lane when a second warp reduces a trailing
// block of its own in the paired kernel).
template <int MT, int G, typename R>
__device__ __forceinline__ void pivot_group(R (&a)[MT], const TriShared<R>& sh, int M,
                                            double* __restrict__ dws, double* __restrict__ ews, const int j)
{
    using C = FastCfg<MT>;
    constexpr int NPR = (8 * G + 8 + 31) / 32;
    constexpr int NP = NPR < C::NW ? NPR : C::NW;
    constexpr unsigned FULL = 0xffffffffu;
    // levels of the shuffle trees: 16 rows sit in half a warp (lanes beyond hold zeros), and with four
    // levels two matrices can share a warp (pack_kernels.cuh)
    constexpr int NSH = (MT <= 16) ? 4 : 5, SH0 = (MT <= 16) ? 8 : 16;
    const int lane = j & 31, warp = j >> 5;
    if (warp >= NP) return;
    const int ihi = (8 * G + 8 < M - 1) ? 8 * G + 8 : M - 1;
    for (int i = ihi; i >= 8 * G + 1; --i) {
        const int k = i - 1 - 8 * G;
        R sigma = sh.red[0];
        if constexpr (NP > 1) sigma += sh.red[1];
        const R alpha = sh.red[4];
        const R xj = sh.xs[j];
        const R praw = dot_blocks<MT, G>(a, sh.xs);
        const R acol = block_pick<MT, G>(a, k);                // A[j][i-1] before the update
        R tau = R(0), scal = R(0), beta = alpha;               // sigma == 0: H_i = I (reading G19)
        if (sigma != R(0)) {
            const R nrm2 = fma(alpha, alpha, sigma);
            const R rinv = rsq(nrm2);
            beta = -copysign(nrm2 * rinv, alpha);
            tau = fma(fabs(alpha), rinv, R(1));                // (beta - alpha) / beta
            scal = R(1) / (alpha - beta);
        }
        const R vj = (j < i - 1) ? xj * scal : ((j == i - 1) ? R(1) : R(0));
        const R pj = (j < i) ? tau * fma(scal, praw, acol) : R(0);
        sh.vbuf[j] = vj;
        sh.pbuf[j] = pj;
        sh.pv[j] = pj * vj;
        if (j < RefLayout<MT>::len(G)) sh.Rf[RefLayout<MT>::base(G) + k * RefLayout<MT>::len(G) + j] = vj;
        if (j == 0) { ews[i - 1] = (double)beta; sh.taus[i] = tau; }
        part_barrier(NP);                                      // ---- B2
        R t = sh.pv[lane];
        if constexpr (NP > 1) t += sh.pv[lane + 32];
        const R nvj = -vj;
#pragma unroll
        for (int step = 0; step < (G + 1 > NSH ? G + 1 : NSH); ++step) {
            if (step < NSH) t += __shfl_xor_sync(FULL, t, SH0 >> step);
            if (step <= G) axpy_block<MT>(a, sh.pbuf, nvj, G - step);
        }
        const R nwj = fma(tau * t, vj, -pj);                   // -(p_j - tau (p.v) v_j)
        axpy_block<MT>(a, sh.vbuf, nwj, G);
        const R xn = block_pick<MT, G>(a, k);                  // A[j][i-1], final: next pivot's x_j
        if (j == i - 1) dws[i - 1] = (double)xn;
        sh.xs[j] = (j < i - 2) ? xn : R(0);
        if (j == i - 2) sh.red[4] = xn;
        R part = (j < i - 2) ? xn * xn : R(0);
#pragma unroll
        for (int step = 0; step < (G > NSH ? G : NSH); ++step) {
            if (step < NSH) part += __shfl_xor_sync(FULL, part, SH0 >> step);
            if (step < G) axpy_block<MT>(a, sh.vbuf, nwj, G - 1 - step);
        }
        if (lane == 0) sh.red[warp] = part;
        part_barrier(NP);                                      // ---- B1 of the next pivot
    }
}

// groups G ... GLO only
template <int MT, int G, int GLO, typename R>
__device__ __forceinline__ void pivot_groups_range(R (&a)[MT], const TriShared<R>& sh, int M,
                                                   double* __restrict__ dws, double* __restrict__ ews, const int j)
{
    pivot_group<MT, G>(a, sh, M, dws, ews, j);
    if constexpr (G > GLO) pivot_groups_range<MT, G - 1, GLO>(a, sh, M, dws, ews, j);
}

template <int MT, int G, typename R>
__device__ __forceinline__ void pivot_groups_down(R (&a)[MT], const TriShared<R>& sh, int M,
                                                  double* __restrict__ dws, double* __restrict__ ews)
{
    pivot_groups_range<MT, G, 0>(a, sh, M, dws, ews, (int)threadIdx.x);
}

// Grid form of the analysis (Procedure 1 lines 1-2,
// Eq.18-19): the local observations of grid point b are gathered from the forecast-observation
// field of the whole periodic grid instead of being read from a materialised Y_loc.
//   local row i = v side^2 + (dy+hw) side + (dx+hw), side = 2 hw + 1, point (y+dy mod Ny, x+dx mod Nx)
//   dY_i = Yf[v][yy][xx][:] - ybar,  d_i = yo[v][yy][xx] - ybar,  r_i = G(dist)/sigma_o^2 (0 if masked)
struct GridArgs {
    const double* Yf;            // [V][Ny][Nx][M]; NULL = not the grid form
    const double* ybar;          // [V][Ny][Nx]   ensemble mean of Yf (Eq.18), formed by grid_obs_mean
    const double* yo;            // [V][Ny][Nx]
    const unsigned char* mask;   // [Ny][Nx] or NULL
    int V, Ny, Nx, hw, loc_kind;
    double L, inv_sig2;
    int point0;                  // grid point of CTA 0
};

// localisation function G of PAPER.md:144: 0 = Gaussian exp(-dist^2/(2 L^2)) (BASELINE.json),
// 1 = Gaspari-Cohn, the 5th-order piecewise rational of ref.[21] with half-width L (zero from 2L)
__host__ __device__ inline double localisation(int kind, double L, double dist)
{
    if (kind == 0) return exp(-(dist * dist) / (2.0 * L * L));
    // Gaspari-Cohn: near branch is even-odd split in u = z^2, 1 - (5/3) u + (5/8) u z + (1/2) u^2 - (1/4) u^2 z;
    // far branch 4 - 5 z + (5/3) u + (5/8) u z - (1/2) u^2 + (1/12) u^2 z - 2 / (3 z)
    const double z = dist / L, u = z * z;
    if (!(z < 2.0)) return 0.0;
    if (z <= 1.0) {
        const double even = fma(u, fma(u, 0.5, -5.0 / 3.0), 1.0);
        const double odd = u * fma(u, -0.25, 0.625);
        return fma(odd, z, even);
    }
    const double even = fma(u, fma(u, -0.5, 5.0 / 3.0), 4.0);
    const double odd = fma(u, fma(u, 1.0 / 12.0, 0.625), -5.0);
    return fma(odd, z, even) - 2.0 / (3.0 * z);
}

// descriptor of local observation row i of grid point (y, x): index of the observed point in the
// [V][Ny][Nx] fields and its weight
__device__ __forceinline__ void grid_row(const GridArgs& g, int y, int x, int i, long& off, double& rloc)
{
    const int side = 2 * g.hw + 1, P2 = side * side;
    const int v = i / P2, rem = i - v * P2;
    const int dy = rem / side - g.hw, dx = rem % side - g.hw;
    int yy = (y + dy) % g.Ny, xx = (x + dx) % g.Nx;
    if (yy < 0) yy += g.Ny;
    if (xx < 0) xx += g.Nx;
    off = ((long)v * g.Ny + yy) * g.Nx + xx;
    const bool seen = !g.mask || g.mask[(long)yy * g.Nx + xx];
    rloc = seen ? localisation(g.loc_kind, g.L, sqrt((double)(dx * dx + dy * dy))) * g.inv_sig2 : 0.0;
}

// Eq.18 for the whole grid: ybar[o] = mean_m Yf[o][m]; one warp per observed point
__global__ void __launch_bounds__(256)
grid_obs_mean(const double* __restrict__ Yf, double* __restrict__ ybar, long nobs, int M)
{
    const long o = (long)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (o >= nobs) return;
    double acc = 0.0;
    for (int m = threadIdx.x & 31; m < M; m += 32) acc += Yf[o * M + m];
    acc = warp_sum(acc);
    if ((threadIdx.x & 31) == 0) ybar[o] = acc / (double)M;
}

// The materialising gather (any M; the path for M > 64 and the cross-check of the fused one):
// Yb[n][p][M], d[n][p], r[n][p] of grid points point0 ... point0+n-1; one CTA per point
__global__ void __launch_bounds__(256)
grid_gather(GridArgs g, int M, int p, double* __restrict__ Yb, double* __restrict__ d, double* __restrict__ r)
{
    const long b = blockIdx.x;
    const int pt = g.point0 + (int)b, y = pt / g.Nx, x = pt - y * g.Nx;
    for (int i = threadIdx.x >> 5; i < p; i += 8) {
        long off; double rl;
        grid_row(g, y, x, i, off, rl);
        const double mean = g.ybar[off];
        for (int m = threadIdx.x & 31; m < M; m += 32) Yb[(b * p + i) * M + m] = g.Yf[off * M + m] - mean;
        if ((threadIdx.x & 31) == 0) { d[b * p + i] = g.yo[off] - mean; r[b * p + i] = rl; }
    }
}

// ---------------------------------------------------------------------------------------------
// a3 for one matrix per CTA.  gram == true: the matrix is not read from A but formed
// from the LETKF inputs (a1, a2: Eq.17 and the right factor of Eq.14) straight into the registers.
// Output: (d, e) in ws.dws / ws.ews, and either (QFORM) the explicit Q = H_{M-1} ... H_1, row-major, in
// Q_, or the reflectors with their taus in ws.refl (RefLayout order, taus behind them) for the
// back-transform in fast_apply.
template <int MT> __host__ __device__ constexpr int refl_doubles() { return RefLayout<MT>::TOTAL + FastCfg<MT>::NT; }

// SPLIT (MT = 64, reflector form): this kernel stops after pivot 33 and hands the trailing 32 x 32
// block (its lower triangle: 528 entries, parked where the reflectors of pivots 32 ... 1 will go),
// the raw pivot column of pivot 32 and its norm to fast_tridiag_tail, one warp per matrix -- so that
// no warp sits at a barrier holding 64 rows' worth of registers while another reduces the last 32
// pivots (ncu, unsplit: barrier stall 1.4 cycles per issue, profiles/r02_ncu_key_metrics.txt).
// The default for 48 < M <= 64 (letkf_set_option("split", 0) restores the one kernel): measured
// 1.07 + 0.25 ms against 1.46 ms for the one kernel (config 3).  The head kernel gets 200 registers
// (LETKF_TRI_REGS64_HEAD, 5 CTAs per SM): at the one kernel's 168 it spills 364 bytes inside the pivot
// loop, whatever shape the hand-over code is given (ptxas), and measures 1.22 ms.
constexpr int SPLIT_LOW = 528, SPLIT_XS = 528, SPLIT_RED = 560;      // offsets inside the first 640 entries

// PAIR (two-warp buckets, reflector form): a CTA reduces TWO matrices.  Pivots M-1 ... 33 need both
// warps (rows 0 ... 63), pivots 32 ... 1 only the warp that holds rows 0 ... 31 -- in the one-matrix
// kernel the other warp then waits at the closing barrier for 36% of the CTA's life (ncu: barrier
// stall 1.4 cycles per issue).  Here both heads run first (the trailing 32 x 32 block of the first
// matrix is parked in shared memory meanwhile), then the two tails run side by side, one per warp,
// each with its own set of broadcast vectors.
constexpr int PAIR_PARK = 32 * 33;
template <int MT, typename R = double, bool PAIR = false> constexpr size_t fast_tridiag_smem_pair()
{
    return fast_tridiag_smem<MT, R>() + (PAIR ? sizeof(R) * (640 + PAIR_PARK + 5 * FastCfg<MT>::NT + 8) : 0);
}

template <int MT, bool GRAM, bool QFORM, typename R = double, bool SPLIT = false, bool PAIR = false>
__global__ void __launch_bounds__(FastCfg<MT>::NT) __maxnreg__((MT == 64) ? ((SPLIT && sizeof(R) == 8) ? LETKF_TRI_REGS64_HEAD : LETKF_TRI_REGS64) : (MT == 48 ? 168 : (MT == 32 ? 128 : 80)))
fast_tridiag(const R* __restrict__ A_, R* __restrict__ Q_, Workspace ws, int M,
                   const double* __restrict__ Yb_, const double* __restrict__ d_,
                   const double* __restrict__ r_, int p, double shift, double* __restrict__ gout_,
                   GridArgs grid, int nbatch)
{
    using C = FastCfg<MT>;
    static_assert(!GRAM || sizeof(R) == sizeof(double), "the Gram step (DMMA) is fp64");
    static_assert(!PAIR || (C::NW == 2 && !QFORM && !SPLIT), "pairs: two-warp buckets, reflector form");
    extern __shared__ __align__(16) unsigned char sm_raw[];
    R* sm = reinterpret_cast<R*>(sm_raw);
    R* tile = sm;
    R* small = sm + RefLayout<MT>::REGION;
    TriShared<R> sh;
    sh.Rf = tile;
    sh.xs = small;
    sh.vbuf = small + C::NT;
    sh.pbuf = small + 2 * C::NT;
    sh.pv = small + 3 * C::NT;
    sh.taus = small + 4 * C::NT;
    sh.red = small + 5 * C::NT;
    R* taus = sh.taus;
    const int j = threadIdx.x, lane = j & 31, warp = j >> 5;
    const int nmat = PAIR ? min(2, nbatch - 2 * (int)blockIdx.x) : 1;
    R* Rf2 = small + 5 * C::NT + 8;                // PAIR: reflectors of the second tail, the parked block, its vectors
    R* park = Rf2 + 640;
    R* small2 = park + PAIR_PARK;
    R a[MT];
#pragma unroll 1
    for (int mi = 0; mi < nmat; ++mi) {
    const size_t b = PAIR ? 2 * (size_t)blockIdx.x + mi : (size_t)blockIdx.x;
    if (PAIR && mi) __syncthreads();               // the shared vectors and the staging tile are free again

    if constexpr (!GRAM) {
        // a_j[c] = A[max(j,c)][min(j,c)] (only the lower triangle is read), 32 rows per pass
        constexpr int HT = RefLayout<MT>::HT;
#pragma unroll
        for (int c = 0; c < MT; ++c) a[c] = R(0);
#pragma unroll
        for (int r0 = 0; r0 < MT; r0 += HT) {
            if (r0 < M) {
                load_rows<MT>(tile, A_ + b * M * M, M, r0, min(HT, M - r0));
                __syncthreads();
#pragma unroll
                for (int c = 0; c < MT; ++c) {
                    if (c < r0 + HT) {                                   // rows beyond this pass: later
                        const int hi = max(j, c), lo = min(j, c);
                        if (hi >= r0 && hi < r0 + HT && hi < M) a[c] = tile[(hi - r0) * C::LDT + lo];
                    }
                }
                __syncthreads();
            }
        }
    } else {
        // a1/a2 on the FP64 tensor cores.  A = shift I + Yb^T diag(r) Yb is a dense contraction
        // over the p local observations, so it runs as mma.sync.m8n8k4.f64 (DMMA): measured on this
        // B200 the instruction reaches the full fp64 rate (37.2 TFLOP/s, the DFMA peak) with 8x fewer
        // issue slots, and the rank-1 DFMA form of this step was issue bound at 35% of peak.
        //   warp w owns rows 32w .. 32w+31 of A: up to 4 row tiles x MT/8 column tiles of 8x8,
        //   64 accumulator doubles per lane (exactly the registers a[] needs afterwards);
        //   the observations are staged 4-row-interleaved, Ys[kk][col][4], so that a fragment
        //   (row i = lane%4 of the k-step, column = 8 tile + lane/4) is 32 consecutive doubles;
        //   the A fragment of row tile rt is the B fragment of column tile rt times r_i.
        const bool gridded = grid.Yf != nullptr;
        const double* Yb = gridded ? nullptr : Yb_ + b * (size_t)p * M;
        const double* dv = gridded ? nullptr : d_ + b * (size_t)p;
        const double* rv = gridded ? nullptr : r_ + b * (size_t)p;
        const int pt = grid.point0 + (int)b, gy = gridded ? pt / grid.Nx : 0, gx = gridded ? pt - gy * grid.Nx : 0;
        constexpr int CT = MT / 8;                                   // column tiles (= row tiles of A)
        constexpr int KBR = (RefLayout<MT>::REGION / MT) / 4 * 4;    // rows the region can stage
        constexpr int RB0 = KBR < 32 ? KBR : 32;
        constexpr int RB = (RB0 < C::NT / 2) ? RB0 : C::NT / 2;      // observation rows per stage (multiple of 4)
        static_assert(RB % 4 == 0 && RB >= 4, "stage size");
        double* Ys = tile;                                           // [RB/4][MT][4]
        double* rloc = sh.xs;                                        // [RB] weight of the staged row
        double* dloc = sh.xs + RB;                                   // [RB] innovation
        double* mloc = sh.vbuf;                                      // [RB] ensemble mean of the row (grid form)
        long*   oloc = reinterpret_cast<long*>(sh.pbuf);             // [RB] observed point of the row (grid form)
        double acc[4][CT][2];
#pragma unroll
        for (int t = 0; t < 4; ++t)
#pragma unroll
            for (int ct = 0; ct < CT; ++ct) { acc[t][ct][0] = 0.0; acc[t][ct][1] = 0.0; }
        double gj = 0.0;
        const int rt0 = 4 * warp;                                    // first row tile of this warp
        for (int i0 = 0; i0 < p; i0 += RB) {
            const int nr = min(RB, p - i0);
            const int nk = (nr + 3) >> 2;                            // k-steps staged (rows padded with r = 0)
            if (j < 4 * nk) {
                double rl = 0.0, dl = 0.0;
                if (j < nr) {
                    if (gridded) {
                        long off;
                        grid_row(grid, gy, gx, i0 + j, off, rl);
                        const double mean = grid.ybar[off];
                        oloc[j] = off; mloc[j] = mean; dl = grid.yo[off] - mean;
                    } else {
                        rl = rv[i0 + j]; dl = dv[i0 + j];
                    }
                }
                rloc[j] = rl; dloc[j] = dl;
            }
            if (gridded) __syncthreads();
            if (j < MT) {                          // thread j stages column j of every row, 8 in flight
                int r = 0;
                for (; r + 8 <= nr; r += 8) {
                    double tmp[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        tmp[u] = (j < M) ? (gridded ? grid.Yf[oloc[r + u] * M + j] - mloc[r + u]
                                                    : Yb[(size_t)(i0 + r + u) * M + j]) : 0.0;
                    double2* y0 = reinterpret_cast<double2*>(Ys + (r >> 2) * (4 * MT) + j * 4);       // r is a multiple of 8:
                    double2* y1 = reinterpret_cast<double2*>(Ys + ((r >> 2) + 1) * (4 * MT) + j * 4); // two whole k-steps
                    y0[0] = make_double2(tmp[0], tmp[1]); y0[1] = make_double2(tmp[2], tmp[3]);
                    y1[0] = make_double2(tmp[4], tmp[5]); y1[1] = make_double2(tmp[6], tmp[7]);
                }
                for (; r < 4 * nk; ++r) {
                    double v = 0.0;
                    if (r < nr && j < M) v = gridded ? grid.Yf[oloc[r] * M + j] - mloc[r] : Yb[(size_t)(i0 + r) * M + j];
                    Ys[(r >> 2) * (4 * MT) + j * 4 + (r & 3)] = v;
                }
            }
            __syncthreads();
            if (j < MT) {                          // a2: g_j += sum_r Yb[r][j] r_r d_r
                for (int kk = 0; kk < nk; ++kk) {
                    const double2* y2 = reinterpret_cast<const double2*>(Ys + kk * (4 * MT) + j * 4);
                    const double2 y01 = y2[0], y23 = y2[1];
                    gj = fma(y01.x, rloc[4 * kk] * dloc[4 * kk], gj);
                    gj = fma(y01.y, rloc[4 * kk + 1] * dloc[4 * kk + 1], gj);
                    gj = fma(y23.x, rloc[4 * kk + 2] * dloc[4 * kk + 2], gj);
                    gj = fma(y23.y, rloc[4 * kk + 3] * dloc[4 * kk + 3], gj);
                }
            }
            if (8 * rt0 < MT) {                    // (a warp beyond the matrix has no tiles: MT = 16 in a 32-thread CTA never gets here)
                for (int kk = 0; kk < nk; ++kk) {
                    const double* base = Ys + kk * (4 * MT) + lane;
                    const double rk = rloc[4 * kk + (lane & 3)];
                    double bfr[CT];
#pragma unroll
                    for (int ct = 0; ct < CT; ++ct) bfr[ct] = base[32 * ct];
#pragma unroll
                    for (int t = 0; t < 4; ++t) {
                        if (8 * (rt0 + t) < MT) {
                            const double afr = base[32 * (rt0 + t)] * rk;   // (= bfr[rt0 + t]; re-read: a run-time
                                                                            // register index would go to local memory)
#pragma unroll
                            for (int ct = 0; ct < CT; ++ct)
                                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                                             : "+d"(acc[t][ct][0]), "+d"(acc[t][ct][1]) : "d"(afr), "d"(bfr[ct]));
                        }
                    }
                }
            }
            __syncthreads();
        }
        // accumulator fragments -> rows in registers: lane l holds A[32w + 8t + l/4][8ct + 2(l%4) + e];
        // each warp passes ITS rows through shared memory, 32 columns at a time (so that no more than
        // 64 doubles are live), and its thread j reads back row j: no block barrier needed.
        constexpr int CH = MT < 32 ? MT : 32;                       // columns per pass
        constexpr int LDC = (MT * (CH + 2) <= RefLayout<MT>::REGION) ? CH + 2 : CH;
        double* cbuf = tile + warp * 32 * LDC;
#pragma unroll
        for (int c0 = 0; c0 < MT; c0 += CH) {
            __syncwarp();
#pragma unroll
            for (int t = 0; t < 4; ++t)
#pragma unroll
                for (int ct = c0 / 8; ct < (c0 + CH) / 8 && ct < CT; ++ct)   // (MT = 48: the last pass is ragged)
                    if (8 * (rt0 + t) < MT)
                        *reinterpret_cast<double2*>(cbuf + (8 * t + (lane >> 2)) * LDC + (8 * ct - c0) + 2 * (lane & 3)) =
                            make_double2(acc[t][ct][0], acc[t][ct][1]);
            __syncwarp();
            if (j < MT) {
                const double2* row2 = reinterpret_cast<const double2*>(cbuf + lane * LDC);
#pragma unroll
                for (int q = 0; q < CH / 2; ++q) {
                    if (c0 + 2 * q + 1 < MT) {                           // MT is even: pairs never straddle the end
                        const double2 v = row2[q];
                        a[c0 + 2 * q] = v.x;
                        a[c0 + 2 * q + 1] = v.y;
                    }
                }
            }
        }
#pragma unroll
        for (int c = 0; c < MT; ++c) a[c] = (j < M && c < M) ? a[c] + ((c == j) ? shift : 0.0) : 0.0;
        __syncthreads();
        if (j < M) gout_[b * M + j] = gj;
    }

    double* dws = ws.dws + b * M;
    double* ews = ws.ews + b * M;
    R* Rf = tile;                                  // reflectors, RefLayout order

    // ---- a3: Householder tridiagonalisation, pivot i = M-1 ... 1, H_i acts on indices 0..i-1.
    // Prologue = the look-ahead of a fictitious pivot M: publish column M-1 and its partial norms.
    {
        const int i0 = M - 1;
        const R x = pick<MT>(a, i0);                   // x_j = A[j][i0]; for j == i0 this is d_i0
        if (j == i0) dws[i0] = (double)x;
        sh.xs[j] = (j < i0 - 1) ? x : R(0);
        if (j == i0 - 1) sh.red[4] = x;
        R part = (j < i0 - 1) ? x * x : R(0);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
        if (lane == 0) sh.red[warp] = part;
        if (j == 0) ews[M - 1] = 0.0;
        __syncthreads();
    }
    // a warp leaves pivot_groups_down when the rows it holds are done (after the B1 that closes
    // the last pivot it took part in), the others carry on with barriers that no longer count it
    if constexpr (SPLIT) {
        static_assert(MT == 64 && !QFORM, "the split form is for the MT = 64 bucket, reflector form");
        pivot_groups_range<MT, (MT - 2) / 8, 4>(a, sh, M, dws, ews, j);
        __syncthreads();
        R* out = reinterpret_cast<R*>(ws.refl + b * ws.reflstride);
        for (int k = RefLayout<MT>::base(4) + j; k < RefLayout<MT>::TOTAL; k += C::NT) out[k] = Rf[k];
        out[RefLayout<MT>::TOTAL + j] = (j >= 33 && j <= M - 1) ? taus[j] : R(0);
        if (j < 32) {
            // row j of the lower triangle at j (j + 1) / 2
            R* low = out + (j * (j + 1)) / 2;
#pragma unroll
            for (int c = 0; c < 32; ++c)
                if (c <= j) low[c] = a[c];
            out[SPLIT_XS + j] = sh.xs[j];
            if (j == 0) { out[SPLIT_RED] = sh.red[0] + sh.red[1]; out[SPLIT_RED + 1] = sh.red[4]; }
        }
        return;
    } else if constexpr (PAIR) {
        pivot_groups_range<MT, (MT - 2) / 8, 4>(a, sh, M, dws, ews, j);
        __syncthreads();
        {   // reflectors of pivots >= 33 and their taus leave now: the region is the next matrix's staging tile
            R* out = reinterpret_cast<R*>(ws.refl + b * ws.reflstride);
            for (int k = RefLayout<MT>::base(4) + j; k < RefLayout<MT>::TOTAL; k += C::NT) out[k] = Rf[k];
            out[RefLayout<MT>::TOTAL + j] = (j >= 33 && j <= M - 1) ? taus[j] : R(0);
        }
        if (mi == 0 && nmat == 2 && j < 32) {      // park the trailing block, the raw pivot column and its norm
#pragma unroll
            for (int c = 0; c < 32; ++c) park[j * 33 + c] = a[c];
            small2[j] = sh.xs[j];
            if (j == 0) { small2[5 * C::NT] = sh.red[0] + sh.red[1]; small2[5 * C::NT + 4] = sh.red[4]; }
        }
        continue;
    } else {
        pivot_groups_down<MT, (MT - 2) / 8>(a, sh, M, dws, ews);
    }
    if constexpr (QFORM) {
        // ---- explicit Q = H_{M-1} ... H_1: thread r owns column r of Q; no synchronisation needed.
        // Column r only needs H_i with i > r, and a warp leaves the loop above exactly when all
        // reflectors with i >= its first row have been stored (barrier 2 of those steps included it),
        // so the upper warps form their columns of Q while warp 0 is still reducing the last 32 rows.
        __syncwarp();
        R (&q)[MT] = a;
#pragma unroll
        for (int c = 0; c < MT; ++c) q[c] = (c == j) ? R(1) : R(0);
        q_groups_up<MT, 0, (MT - 2) / 8>(q, static_cast<const R*>(Rf), static_cast<const R*>(taus), M, warp * 4);
        if (j < M) {
            R* Q = Q_ + b * M * M;
#pragma unroll
            for (int c = 0; c < MT; ++c)
                if (c < M) Q[(size_t)c * M + j] = q[c];
        }
    } else {
        __syncthreads();
        // reflectors (RefLayout order; H_i with i >= M are never read) and taus for the back-transform
        R* out = reinterpret_cast<R*>(ws.refl + b * ws.reflstride);
        for (int k = j; k < RefLayout<MT>::TOTAL; k += C::NT) out[k] = Rf[k];
        out[RefLayout<MT>::TOTAL + j] = (j >= 1 && j <= M - 1) ? taus[j] : R(0);
    }
    }   // matrices of the CTA
    if constexpr (PAIR) {
        // ---- the tails: pivots min(32, M-1) ... 1, one matrix per warp
        __syncthreads();
        const size_t b0 = 2 * (size_t)blockIdx.x;
        size_t bt = b0;
        TriShared<R> st = sh;
        if (nmat == 2) {
            if (warp == 1) {                       // the first matrix: its block comes back from the park
                st.Rf = Rf2;
                st.xs = small2; st.vbuf = small2 + C::NT; st.pbuf = small2 + 2 * C::NT; st.pv = small2 + 3 * C::NT;
                st.taus = small2 + 4 * C::NT; st.red = small2 + 5 * C::NT;
#pragma unroll
                for (int c = 0; c < 32; ++c) a[c] = park[lane * 33 + c];
            } else {
                bt = b0 + 1;                       // the second matrix is still in warp 0's registers
                if (lane == 0) st.red[0] += st.red[1];
            }
        } else {
            if (warp == 1) return;
            if (lane == 0) st.red[0] += st.red[1];
        }
        __syncwarp();
        pivot_groups_range<MT, 3, 0>(a, st, M, ws.dws + bt * M, ws.ews + bt * M, lane);
        __syncwarp();
        R* out = reinterpret_cast<R*>(ws.refl + bt * ws.reflstride);
        for (int k = lane; k < 640; k += 32) out[k] = st.Rf[k];
        if (lane >= 1) out[RefLayout<MT>::TOTAL + lane] = st.taus[lane];
        if (lane == 0 && M > 32) out[RefLayout<MT>::TOTAL + 32] = st.taus[32];
    }
}

// Trailing 32 x 32 problem of the split form: pivots 32 ... 1, one warp per matrix (FastCfg<32>).
template <typename R>
__global__ void __maxnreg__(128)
fast_tridiag_tail(Workspace ws, int M)
{
    constexpr int MT = 32;
    extern __shared__ __align__(16) unsigned char sm_raw[];
    R* sm = reinterpret_cast<R*>(sm_raw);
    TriShared<R> sh;
    sh.Rf = sm;                                  // groups 0..3: 640 entries
    R* small = sm + 640;
    sh.xs = small; sh.vbuf = small + 32; sh.pbuf = small + 64; sh.pv = small + 96;
    sh.taus = small + 128;                       // [40]
    sh.red = small + 168;                        // [8]
    const int j = threadIdx.x;
    const size_t b = blockIdx.x;
    R* io = reinterpret_cast<R*>(ws.refl + b * ws.reflstride);
    R a[MT];
#pragma unroll
    for (int c = 0; c < MT; ++c) {
        const int hi = c > j ? c : j, lo = c > j ? j : c;
        a[c] = io[(hi * (hi + 1)) / 2 + lo];
    }
    sh.xs[j] = io[SPLIT_XS + j];
    if (j == 0) { sh.red[0] = io[SPLIT_RED]; sh.red[4] = io[SPLIT_RED + 1]; }
    __syncwarp();
    // as a 33 x 33 problem whose last column is already in xs: pivot 32 takes it from there
    pivot_groups_down<MT, 3>(a, sh, 33, ws.dws + b * M, ws.ews + b * M);
    __syncwarp();
    for (int k = j; k < 640; k += 32) io[k] = sh.Rf[k];
    constexpr int TOT64 = RefLayout<64>::TOTAL;
    io[TOT64 + j] = (j >= 1) ? sh.taus[j] : R(0);
    if (j == 0) io[TOT64 + 32] = sh.taus[32];
}
template <typename R> constexpr size_t fast_tridiag_tail_smem() { return sizeof(R) * (640 + 176); }

// ---------------------------------------------------------------------------------------------
// a5: V = Q Z = H_{M-1} ... H_1 Z.  Z is the product of the logged rotations: thread r replays
// them on row r of the identity held in registers; the matrix is then turned through shared
// memory so that thread k holds eigenvector k of T, to which it applies the reflectors (q_group:
// dot product and update inside the thread, reflectors as 16-byte broadcast loads).
// Dynamic shared memory: A region [ap_a_doubles], reflectors + taus [refl_doubles], hdr[swcap] u32,
// inv[MT] int (+ the epilogue's arrays, which alias the reflectors once they are applied).
constexpr int AP_S = 8;      // sweeps staged per barrier round (measured: 2 / 4 / 8 -> 2.05 / 1.99 / 1.93 ms)
// A region of fast_apply: the staged rotations [2][AP_S][MT] double2, later the 32 x 33 tiles of
// the transposition (one per warp) and of the output pass (HT padded rows)
template <int MT> __host__ __device__ constexpr int ap_a_doubles()
{
    constexpr int cs = 4 * AP_S * MT, tr = FastCfg<MT>::NW * 32 * 33, out = (MT < 32 ? MT : 32) * (MT + 1);
    constexpr int m1 = cs > tr ? cs : tr, m2 = m1 > out ? m1 : out;
    return (m2 + 1) & ~1;
}
// a6-a9 fused into the tail of fast_apply (the analysis call when W is not wanted): V never
// goes to HBM.  lam = eigenvalues ascending (output order), g = Yb^T (r o d), Eq.14.
struct EpiArgs {
    const double* lam;    // [n][M]
    const double* g;      // [n][M]
    const double* Xb;     // [n][ns][M]
    double*       Xa;     // [n][ns][M]
    double*       wbar;   // [n][M] or NULL
    int           ns;
};
constexpr int EPI_NS_MAX = 15;     // fused epilogue for nstate <= 15, generic_epilogue beyond
// doubles the epilogue needs: Bm[MT][ns+1 padded to even], Tm[ns+1][MT], xbar[ns], cvec[ns], red[NW][ns]; they alias
// the reflector region, which is enlarged when they do not fit
template <int MT> __host__ __device__ inline int fast_epi_doubles(int ns)
{
    return MT * ((ns + 2) & ~1) + MT * (ns + 1) + 2 * ns + FastCfg<MT>::NW * ns + 4;
}
// words of the header region of fast_apply: the sweep headers of the replay, or (eigenvector path)
// ds[MT], es[MT], lam sorted [MT] as doubles and perm [MT] as bytes
template <int MT> __host__ __device__ inline int ap_hdr_words(int swcap)
{
    const int gv = 6 * MT + MT / 4 + 8;
    return swcap > gv ? swcap : gv;
}

template <int MT> __host__ __device__ inline int fast_apply_rd(int epi_ns, bool qform)
{
    int rd = qform ? 0 : refl_doubles<MT>();
    if (epi_ns > 0 && fast_epi_doubles<MT>(epi_ns) > rd) rd = (fast_epi_doubles<MT>(epi_ns) + 1) & ~1;
    return rd;
}
template <int MT> size_t fast_apply_smem(int swcap, int epi_ns, bool qform)
{
    const int rd = fast_apply_rd<MT>(epi_ns, qform);
    return sizeof(double) * ((size_t)ap_a_doubles<MT>() + rd) + sizeof(uint32_t) * (size_t)ap_hdr_words<MT>(swcap) + sizeof(int) * MT + 16;
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src)
{
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all()
{
    asm volatile("cp.async.wait_all;" ::: "memory");
}

// ---- one contiguous record global -> shared by the TMA unit (cp.async.bulk, SASS UBLKCP): one thread arms an
// mbarrier with the byte count and issues the copy, no thread spends an instruction per 16 bytes; whoever needs the
// data waits for the barrier's phase.  Addresses and size are multiples of 16 bytes.
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(a), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gmem_src, unsigned bytes, unsigned long long* bar)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar), d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(a), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(d), "l"(gmem_src), "r"(bytes), "r"(a) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    unsigned ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    } while (!ok);
}

// Rotations i = m-1 ... lo on columns (i, i+1):  f = z[i+1]; z[i+1] = s z[i] + c f; z[i] = c z[i] - s f.
// Blocks of 4 rotations, entered at the block of m-1 and left after the block of lo; cs[] holds
// the identity (1, 0) outside [lo, m), so the overhang at both ends changes nothing.  The only
// dependent chain from one rotation to the next is the single FMA that produces z[i].
template <int MT, typename R>
__device__ __forceinline__ void apply_sweep(R (&z)[MT], const double2* cs, int lo, int m)
{
    switch ((m - 1) >> 2) {
#define LETKF_ROT1(i, t)                                                      \
        if constexpr ((i) + 1 < MT) {                                         \
            const R f = z[(i) + 1];                                           \
            const R zi = z[i];                                                \
            const R tc = (R)t.x, ts = (R)t.y;                                 \
            z[(i) + 1] = fma(ts, zi, tc * f);                                 \
            z[i] = fma(-ts, f, tc * zi);                                      \
        }
#define LETKF_ROT(g)                                                          \
    case g:                                                                   \
        if constexpr (4 * (g) + 3 < MT) {                                     \
            const double2 t3 = cs[4 * (g) + 3], t2 = cs[4 * (g) + 2];         \
            const double2 t1 = cs[4 * (g) + 1], t0 = cs[4 * (g)];             \
            LETKF_ROT1(4 * (g) + 3, t3) LETKF_ROT1(4 * (g) + 2, t2)           \
            LETKF_ROT1(4 * (g) + 1, t1) LETKF_ROT1(4 * (g), t0)               \
            if (4 * (g) <= lo) break;                                         \
        }
        LETKF_ROT(15) LETKF_ROT(14) LETKF_ROT(13) LETKF_ROT(12) LETKF_ROT(11) LETKF_ROT(10) LETKF_ROT(9)
        LETKF_ROT(8) LETKF_ROT(7) LETKF_ROT(6) LETKF_ROT(5) LETKF_ROT(4) LETKF_ROT(3) LETKF_ROT(2)
        LETKF_ROT(1) LETKF_ROT(0)
#undef LETKF_ROT
#undef LETKF_ROT1
    }
}

// 32 x 32 block moves of the transposition (compile-time register offsets)
template <int MT, int C0, typename R>
__device__ __forceinline__ void tr_put(const R (&z)[MT], R* T, int lane)
{
#pragma unroll
    for (int c = 0; c < 32; ++c)
        if (C0 + c < MT) T[lane * 33 + c] = z[C0 + c];
}
template <int MT, int R0, typename R>
__device__ __forceinline__ void tr_get(R (&z)[MT], const R* T, int lane)
{
#pragma unroll
    for (int rr = 0; rr < 32; ++rr)
        if (R0 + rr < MT) z[R0 + rr] = T[rr * 33 + lane];
}
// Thread t holds row t of an MT x MT matrix (threads t >= MT: nothing that matters); afterwards
// thread t holds column t (an involution: the same call turns it back).  One 32 x 33 tile per warp;
// with two warps the diagonal blocks turn inside their warp and the two off-diagonal blocks swap
// through both tiles at once, so a thread never holds more than its MT values.
template <int MT, typename R>
__device__ __forceinline__ void transpose_regs(R (&z)[MT], R* tiles)
{
    constexpr int NW = FastCfg<MT>::NW;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    R* T = tiles + warp * (32 * 33);
    if constexpr (NW == 1) {
        __syncwarp();
        tr_put<MT, 0>(z, T, lane);
        __syncwarp();
        tr_get<MT, 0>(z, T, lane);
        __syncwarp();
    } else {
        static_assert(NW == 2, "at most two warps per matrix");
        __syncthreads();                                   // the tiles are free
        if (warp == 0) tr_put<MT, 0>(z, T, lane); else tr_put<MT, 32>(z, T, lane);
        __syncwarp();
        if (warp == 0) tr_get<MT, 0>(z, T, lane); else tr_get<MT, 32>(z, T, lane);
        __syncwarp();
        // warp 0 hands block (rows 0..31, columns 32..) to warp 1, warp 1 block (rows 32.., columns 0..31) to warp 0
        if (warp == 0) tr_put<MT, 32>(z, T, lane); else tr_put<MT, 0>(z, T, lane);
        __syncthreads();
        const R* O = tiles + (1 - warp) * (32 * 33);
        if (warp == 0) tr_get<MT, 32>(z, O, lane); else tr_get<MT, 0>(z, O, lane);
        __syncthreads();
    }
}

// 1/x to about an ulp: hardware seed (2^-23) and two Newton steps; x normal, non-zero
__device__ __forceinline__ double fast_rcp(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double t = fma(-x, y, 1.0);
    y = fma(y, t, y);
    t = fma(-x, y, 1.0);
    return fma(y, t, y);
}

// Eigenvector of the symmetric tridiagonal T (diagonal ds, off-diagonal es with the negligible
// entries set to exactly 0, so T is a direct sum of unreduced blocks) for the eigenvalue lam of
// the block [lo, hi], by the twisted factorisation of T - lam I (Fernando; Parlett & Dhillon: the
// "getvec" step of MRRR applied to T itself): with the pivots D+ of L D+ L^T from the top and D- of
// U D- U^T from the bottom, gamma_i = D+_i + D-_i - (d_i - lam) is the one non-zero residual
// component of the vector that solves the equations twisted at i, so the twist goes where |gamma|
// is smallest and  z_r = 1,  z_i = -(e_i / D+_i) z_{i+1} (i < r),  z_{i+1} = -(e_i / D-_{i+1}) z_i (i >= r).
// One thread per eigenvector, everything in registers with compile-time indices (the loops run
// over all MT indices: outside the block e = 0 restarts the recurrences and zeroes the vector).
// z doubles as the store of the reciprocal pivots until each entry is final.  Returns the
// eigenvector, normalised, and its residual norm ||(T - lam) z||_2.
template <int MT>
__device__ __forceinline__ double getvec(double (&z)[MT], const double* ds, const double* es, double lam,
                                         int lo, int hi, double pivmin)
{
    // forward pivots: z[i] = 1 / D+_i
    {
        double P = ds[0] - lam;
#pragma unroll
        for (int i = 0; i < MT; ++i) {
            P = (fabs(P) < pivmin) ? -pivmin : P;
            z[i] = fast_rcp(P);
            if (i + 1 < MT) { const double ei = es[i]; P = fma(-(ei * ei), z[i], ds[i + 1] - lam); }
            if ((i & 7) == 7) __syncwarp();        // scheduling fence: ptxas does not hoist shared loads across it
        }
    }
    // backward pivots on the fly: the twist index
    int r = lo;
    {
        double best = 1.7976931348623157e308;
        double Dm = ds[MT - 1] - lam;
#pragma unroll
        for (int i = MT - 1; i >= 0; --i) {
            Dm = (fabs(Dm) < pivmin) ? -pivmin : Dm;
            const double di = ds[i] - lam;
            double Pi = di;
            if (i > 0) { const double el = es[i - 1]; Pi = fma(-(el * el), z[i - 1], di); }
            Pi = (fabs(Pi) < pivmin) ? -pivmin : Pi;
            const double gam = fabs(Pi + Dm - di);
            if (i >= lo && i <= hi && gam < best) { best = gam; r = i; }
            if (i > 0) { const double el = es[i - 1]; Dm = fma(-(el * el), fast_rcp(Dm), ds[i - 1] - lam); }
            if ((i & 7) == 0) __syncwarp();
        }
    }
    // from the bottom down to the twist: 1 / D-_i into z[i] (i > r); below the twist the vector itself
    {
        double Dm = ds[MT - 1] - lam, zc = 1.0;
#pragma unroll
        for (int i = MT - 1; i >= 0; --i) {
            if (i > r) {
                Dm = (fabs(Dm) < pivmin) ? -pivmin : Dm;
                const double rd = fast_rcp(Dm);
                z[i] = rd;
                if (i > 0) { const double el = es[i - 1]; Dm = fma(-(el * el), rd, ds[i - 1] - lam); }
            } else if (i == r) {
                z[i] = 1.0;
            } else {
                zc = -(es[i] * z[i]) * zc;
                z[i] = zc;
            }
            if ((i & 7) == 0) __syncwarp();
        }
    }
    // from the twist up
    {
        double zc = 1.0;
#pragma unroll
        for (int i = 0; i + 1 < MT; ++i) {
            if (i >= r) {
                zc = -(es[i] * z[i + 1]) * zc;
                z[i + 1] = zc;
            }
            if ((i & 7) == 7) __syncwarp();
        }
    }
    double n0 = 0.0, n1 = 0.0;
#pragma unroll
    for (int i = 0; i + 1 < MT; i += 2) { n0 = fma(z[i], z[i], n0); n1 = fma(z[i + 1], z[i + 1], n1); }
    const double sc = rsqrt(n0 + n1);
    double r0 = 0.0, r1 = 0.0, zm = 0.0;
#pragma unroll
    for (int i = 0; i < MT; ++i) {
        z[i] *= sc;
        // residual row i - 1 is complete once z[i] is known
        if (i > 0) {
            const double up = (i > 1) ? es[i - 2] * zm : 0.0;
            const double t = fma(ds[i - 1] - lam, z[i - 1], fma(es[i - 1], z[i], up));
            if (i & 1) r0 = fma(t, t, r0); else r1 = fma(t, t, r1);
        }
        if (i > 0) zm = z[i - 1];
        if ((i & 7) == 7) __syncwarp();
    }
    {
        const double up = (MT > 1) ? es[MT - 2] * z[MT - 2] : 0.0;
        const double t = fma(ds[MT - 1] - lam, z[MT - 1], up);
        r0 = fma(t, t, r0);
    }
    return sqrt(r0 + r1);
}

// The eigenvectors of T of matrix b without a single rotation (route FLAG_GETVEC of fast_apply):
// thread k = position k, its eigenvalue is w[inv[k]]; on return z holds eigenvector k (a unit vector
// for a 1 x 1 block).  `scratch` holds ap_hdr_words<MT>() words, `vbuf` 32 (MT + 1) doubles.  Called
// by all threads of the CTA (barriers inside); returns false when a residual is suspicious and the
// matrix has to go to the classic iteration.
template <int MT>
__device__ __forceinline__ bool direct_eigenvectors(double (&z)[MT], uint32_t* scratch, double* vbuf, const Workspace& ws,
                                                    const double* __restrict__ w_, size_t b, int M, const int* inv)
{
    using C = FastCfg<MT>;
    const int r = threadIdx.x;
    bool ok;
    double*        ds    = reinterpret_cast<double*>(scratch);         // [MT]
    double*        es    = ds + MT;                                // [MT] negligible entries are exactly 0
    double*        wsrt  = es + MT;                                // [MT] eigenvalues ascending
    unsigned char* perm8 = reinterpret_cast<unsigned char*>(wsrt + MT);   // [MT] position of the k-th smallest
    unsigned*      cutw  = reinterpret_cast<unsigned*>(perm8 + MT);       // [2] bit i: block boundary behind i
    if (r < MT) {
        ds[r] = (r < M) ? ws.dws[b * M + r] : 0.0;
        es[r] = (r < M - 1) ? ws.ews[b * M + r] : 0.0;
        wsrt[r] = (r < M) ? w_[b * M + r] : 0.0;
        perm8[r] = (unsigned char)((r < M) ? ws.perm[b * M + r] : r);
    }
    __syncthreads();
    // the threshold and the split of ql_log_kernel, on the same numbers
    const double eps = 1.1102230246251565e-16;
    // (max is exact in any order: the same number the QL kernel's serial loop finds)
    double nrm = (r < M) ? fabs(ds[r]) + (r < M - 1 ? fabs(es[r]) : 0.0) : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nrm = fmax(nrm, __shfl_xor_sync(0xffffffffu, nrm, o));
    double* nrmw = reinterpret_cast<double*>(cutw + 2);                      // [2]
    if ((r & 31) == 0) nrmw[r >> 5] = nrm;
    __syncthreads();
    if constexpr (C::NW > 1) nrm = fmax(nrmw[0], nrmw[1]);
    const double thr = eps * nrm;
    bool cut = true;
    if (r < M - 1) cut = fabs(es[r]) <= fmax(eps * (fabs(ds[r]) + fabs(ds[r + 1])), GV_SPLIT * thr);
    __syncthreads();
    if (r < MT && cut) es[r] = 0.0;
    const unsigned cw = __ballot_sync(0xffffffffu, cut);
    if ((r & 31) == 0) cutw[r >> 5] = cw;
    __syncthreads();
    int lo = 0, hi = M - 1;
    double lam = 0.0;
    if (r < M) {
        const unsigned long long cuts = (C::NW > 1) ? ((unsigned long long)cutw[1] << 32 | cutw[0]) : (unsigned long long)cutw[0];
        const unsigned long long below = cuts & ((1ull << r) - 1ull);        // boundaries behind indices < r
        lo = below ? 64 - __clzll((long long)below) : 0;
        const unsigned long long above = cuts >> r;                          // bit 0: boundary behind r
        hi = above ? r + __ffsll((long long)above) - 1 : M - 1;
        if (hi > M - 1) hi = M - 1;
        lam = wsrt[inv[r]];
    }
    // (every thread runs it -- the fences inside want whole warps; a 1 x 1 block gets its unit vector)
    const bool own = r < M && lo < hi;
    double res = getvec<MT>(z, ds, es, lam, lo, hi, fmax(thr * eps, 1e-300));
    if (!own) {
        res = 0.0;
#pragma unroll
        for (int c = 0; c < MT; ++c) z[c] = (c == r) ? 1.0 : 0.0;
    }
    // anything suspicious hands the matrix to the classic iteration below
    const bool bad = !(res <= 64.0 * eps * nrm * sqrt((double)M));
    if (__syncthreads_or(bad ? 1 : 0)) {
        ok = false;
    } else {
        ok = true;
        // eigenvalues closer than GV_GAP ||T|| inside a block: first-order symmetric orthogonalisation,
        // z_k -= 1/2 (z_q . z_k) z_q for every such partner q (the classifier bounds their number);
        // the vectors pass through shared memory 32 at a time
        const double gapabs = GV_GAP * nrm;
        PartnerList pl;                                                 // same-block eigenvalues within GV_GAP ||T|| (the classifier bounds them)
        if (own) {
            const int s0 = inv[r];
            for (int t = 1; s0 - t >= 0 && lam - wsrt[s0 - t] < gapabs; ++t) {
                const int q = perm8[s0 - t];
                if (q >= lo && q <= hi) pl.add(q);
            }
            for (int t = 1; s0 + t < M && wsrt[s0 + t] - lam < gapabs; ++t) {
                const int q = perm8[s0 + t];
                if (q >= lo && q <= hi) pl.add(q);
            }
        }
        if (__syncthreads_or(pl.np)) {
            constexpr int LDV = MT + 1;
            const int npw = __reduce_max_sync(0xffffffffu, pl.np);             // whole warps walk the longest list
#pragma unroll 1
            for (int ph = 0; ph < C::NW; ++ph) {
                if (ph) __syncthreads();
                if ((r >> 5) == ph) {
#pragma unroll
                    for (int i = 0; i < MT; ++i) vbuf[(r & 31) * LDV + i] = z[i];
                }
                __syncthreads();
#pragma unroll 1
                for (int t = 0; t < npw; ++t) {
                    const int q = pl.get(t);
                    const bool act = t < pl.np && (q >> 5) == ph;
                    const double* vq = vbuf + (act ? (q & 31) : 0) * LDV;
                    double d0 = 0.0, d1 = 0.0;
#pragma unroll
                    for (int i = 0; i + 1 < MT; i += 2) {
                        d0 = fma(z[i], vq[i], d0); d1 = fma(z[i + 1], vq[i + 1], d1);
                        if ((i & 7) == 6) __syncwarp();
                    }
                    const double h = act ? -0.5 * (d0 + d1) : 0.0;
#pragma unroll
                    for (int i = 0; i < MT; ++i) {
                        z[i] = fma(h, vq[i], z[i]);
                        if ((i & 7) == 7) __syncwarp();
                    }
                }
            }
        }
    }
    return ok;
}

template <int MT, bool EPI, bool QFORM>
__global__ void __launch_bounds__(FastCfg<MT>::NT, (MT == 64) ? 6 : (MT == 48 ? LETKF_AP48 : 16))
fast_apply(double* __restrict__ V_, double* __restrict__ w_, int* __restrict__ info_, Workspace ws, int M, EpiArgs ep)
{
    using C = FastCfg<MT>;
    extern __shared__ __align__(16) double sm[];
    double*   areg = sm;                                   // A region
    double2*  cs   = reinterpret_cast<double2*>(sm);       // [2][AP_S][MT] while rotating
    double*   R    = sm + ap_a_doubles<MT>();              // reflectors, RefLayout order
    double*   taus = R + RefLayout<MT>::TOTAL;
    const int rd = fast_apply_rd<MT>(EPI ? ep.ns : 0, QFORM);
    uint32_t* hdr  = reinterpret_cast<uint32_t*>(R + rd);
    int*      inv  = reinterpret_cast<int*>(hdr + ap_hdr_words<MT>(ws.swcap));
    const int r = threadIdx.x;
    const size_t b = blockIdx.x;
    const int flag = ws.flags[b];
    const bool direct = !QFORM && flag == FLAG_GETVEC;     // eigenvectors of T by twisted factorisations
    bool flagged = flag == FLAG_SLOW;                      // rotation log unusable: classic QL below
    const int nsw = (flag == FLAG_REPLAY) ? ws.nsweeps[b] : 0;
    const double2* rot = ws.rot + b * ws.logcap;

    constexpr int HT = MT < 32 ? MT : 32;          // rows per pass through the tile
    double* tile = areg;
    for (int s = r; s < nsw; s += C::NT) hdr[s] = ws.hdr[b * ws.swcap + s];
    if (!flagged && r < M) inv[ws.perm[b * M + r]] = r;    // output column of QL-order column c
    double z[MT];
    __shared__ unsigned long long refl_bar;
    if constexpr (!QFORM) {
        // the reflectors fly in while the eigenvectors of T are formed: one bulk copy of the record by the TMA unit
        if (r == 0) {
            mbar_init(&refl_bar, 1);
            bulk_load(R, ws.refl + b * ws.reflstride, (unsigned)(sizeof(double) * refl_doubles<MT>()), &refl_bar);
        }
    }
    bool columns = false;                          // z holds a column of Z (an eigenvector of T) rather than a row

    if (direct) {
        // ---- eigenvectors of T by twisted factorisations (the reflectors keep flying in meanwhile)
        if (direct_eigenvectors<MT>(z, hdr, areg, ws, w_, b, M, inv)) columns = true;
        else flagged = true;
        cp_async_wait_all();
        __syncthreads();
    } else if (!flagged) {
        if constexpr (QFORM) {
            // row r of Q (stored by fast_tridiag in the output buffer) through the tile, HT rows per pass
            const double* Q = V_ + b * M * M;
#pragma unroll
            for (int c = 0; c < MT; ++c) z[c] = 0.0;
#pragma unroll
            for (int r0 = 0; r0 < MT; r0 += HT) {
                if (r0 < M) {
                    load_rows<MT>(tile, Q, M, r0, min(HT, M - r0));
                    __syncthreads();
                    if (r >= r0 && r < r0 + HT && r < M) {
#pragma unroll
                        for (int c = 0; c < MT; ++c) z[c] = (c < M) ? tile[(r - r0) * C::LDT + c] : 0.0;
                    }
                    __syncthreads();
                }
            }
        } else {
#pragma unroll
            for (int c = 0; c < MT; ++c) z[c] = (c == r) ? 1.0 : 0.0;
            __syncthreads();
        }
        // The (c, s) of AP_S sweeps are staged per barrier round, double-buffered: thread r copies the
        // rotation that acts on columns (r, r+1) of each sweep straight from the log into shared
        // memory (cp.async, no registers), identity outside [lo, m); the copies of round k+1 fly
        // while round k is applied.
        int spos = 0;                                   // log position of the next sweep to stage
        auto stage = [&](int round) {
            double2* dst = cs + (round & 1) * AP_S * MT;
#pragma unroll
            for (int t = 0; t < AP_S; ++t) {
                const int s = round * AP_S + t;
                if (s < nsw) {
                    const uint32_t h = hdr[s];
                    const int lo = h & 0xffff, m = h >> 16;
                    if (r < MT) {
                        if (r >= lo && r < m) cp_async16(dst + t * MT + r, rot + spos + (m - 1 - r));
                        else dst[t * MT + r] = make_double2(1.0, 0.0);
                    }
                    spos += m - lo;
                }
            }
        };
        const int nrounds = (nsw + AP_S - 1) / AP_S;
        if (nrounds > 0) stage(0);
        cp_async_wait_all();
        __syncthreads();
        for (int k = 0; k < nrounds; ++k) {
            if (k + 1 < nrounds) stage(k + 1);
            const double2* cur = cs + (k & 1) * AP_S * MT;
            const int send = min(nsw, (k + 1) * AP_S);
#pragma unroll 1
            for (int s = k * AP_S; s < send; ++s) {
                const uint32_t h = hdr[s];
                apply_sweep<MT>(z, cur + (s - k * AP_S) * MT, h & 0xffff, h >> 16);
            }
            cp_async_wait_all();
            __syncthreads();
        }
    }
    if (flagged) {
        // Slow path (LETKF_INFO_SLOWPATH): the classic iteration, one sweep at a time -- thread 0 runs
        // the recurrences of ql_next_sweep (which treats underflow, overflow and NaN case by case) on
        // the tridiagonal form the reduction left, all threads apply the sweep to their rows.
        double*  dsm  = areg;                                        // [MT]
        double*  esm  = areg + MT;                                   // [MT]
        double2* sink = reinterpret_cast<double2*>(areg + 2 * MT);   // [MT] in generation order
        double2* csb  = sink + MT;                                   // [MT] by column, identity outside [lo, m)
        int*     ctl  = reinterpret_cast<int*>(csb + MT);            // rc, lo, m, fail
        __syncthreads();
        if constexpr (QFORM) {
            const double* Q = V_ + b * M * M;                        // row r of Q straight from global memory
#pragma unroll
            for (int c = 0; c < MT; ++c) z[c] = (r < M && c < M) ? Q[(size_t)r * M + c] : 0.0;
        } else {
#pragma unroll
            for (int c = 0; c < MT; ++c) z[c] = (c == r) ? 1.0 : 0.0;
        }
        if (r < M) { dsm[r] = ws.dws[b * M + r]; esm[r] = ws.ews[b * M + r]; }
        __syncthreads();
        QLState st{0, 0, 0, 0.0};
        if (r == 0) { esm[M - 1] = 0.0; st.thr = ql_threshold(dsm, esm, 1, M); }
        for (;;) {
            if (r == 0) {
                int lo = 0, m = 0;
                ctl[0] = ql_next_sweep(st, dsm, esm, 1, M, sink, M, lo, m);
                ctl[1] = lo; ctl[2] = m;
            }
            __syncthreads();
            if (ctl[0] != 1) break;
            const int lo = ctl[1], m = ctl[2];
            if (r < MT) csb[r] = (r >= lo && r < m) ? sink[m - 1 - r] : make_double2(1.0, 0.0);
            __syncthreads();
            apply_sweep<MT>(z, csb, lo, m);
            __syncthreads();
        }
        int* permsm = reinterpret_cast<int*>(sink);                  // the sink is free now
        if (r == 0) { sort_eigenvalues(dsm, 1, permsm, 1, M); ctl[3] = st.fail; }
        __syncthreads();
        if (r < M) { inv[permsm[r]] = r; w_[b * M + r] = dsm[r]; }
        if (r == 0 && info_) info_[b] = ctl[3] | 0x40000000;
        cp_async_wait_all();
        __syncthreads();
    }

    if constexpr (!QFORM) {
        // rows of Z -> eigenvectors of T: thread k holds column k (QL order); then V = H_{M-1} ... H_1 Z
        if (!columns) transpose_regs<MT>(z, areg);
        mbar_wait(&refl_bar, 0);                   // (every path here has passed a block barrier since the copy was issued)
        q_groups_up<MT, 0, (MT - 2) / 8>(z, R, taus, M, 0);
    }

    if constexpr (!EPI && QFORM) {
        // sorted, row-major V through the tile, HT rows per pass (thread r holds row r)
        double* V = V_ + b * M * M;
#pragma unroll
        for (int r0 = 0; r0 < MT; r0 += HT) {
            if (r0 < M) {
                if (r >= r0 && r < r0 + HT && r < M) {
#pragma unroll
                    for (int c = 0; c < MT; ++c)
                        if (c < M) tile[(r - r0) * C::LDT + inv[c]] = z[c];
                }
                __syncthreads();
                if (r < M) {                       // thread r writes column r of every row: coalesced
                    const int nr = min(HT, M - r0);
#pragma unroll 8
                    for (int rr = 0; rr < nr; ++rr) V[(size_t)(r0 + rr) * M + r] = tile[rr * C::LDT + r];
                }
                __syncthreads();
            }
        }
    } else if constexpr (!EPI) {
        // sorted, row-major V through the tile, HT rows per pass: thread k scatters its column into
        // output column inv[k], thread t then writes column t of every row (coalesced)
        double* V = V_ + b * M * M;
        const int oc = (r < M) ? inv[r] : 0;
#pragma unroll
        for (int r0 = 0; r0 < MT; r0 += HT) {
            if (r0 < M) {
                __syncthreads();
                if (r < M) {
#pragma unroll
                    for (int rr = 0; rr < HT; ++rr)
                        if (r0 + rr < MT) tile[rr * C::LDT + oc] = z[r0 + rr];
                }
                __syncthreads();
                if (r < M) {
                    const int nr = min(HT, M - r0);
#pragma unroll 8
                    for (int rr = 0; rr < nr; ++rr) V[(size_t)(r0 + rr) * M + r] = tile[rr * C::LDT + r];
                }
            }
        }
    } else {
        if constexpr (QFORM) transpose_regs<MT>(z, areg);                    // rows of V -> eigenvectors
        // ---- a6-a9 on the V held in registers (thread k = eigenvector k in QL order, its eigenvalue
        // lam_k = lam[inv[k]]; sums over k do not care about the order).
        //   T[q][k] = sum_r V[r][k] B[r][q],  B = [g | dX^T]     (inside the thread)
        //   t'_k = T[0][k]/lam_k,  U'[s][k] = sqrt(M-1) T[1+s][k]/sqrt(lam_k)
        //   c_s = sum_k T[1+s][k] t'_k  (= dX_s . wbar)
        // then the matrix is turned back (thread m = row m of V) for
        //   wbar_m = sum_k V[m][k] t'_k,   Xa[s][m] = xbar_s + c_s + sum_k U'[s][k] V[m][k]
        const int ns = ep.ns, nq = ns + 1, nqp = (nq + 1) & ~1;             // rows of Bm padded to whole pairs
        __syncthreads();                                                    // the reflectors are dead
        double* Bm   = R;                                                   // [MT][nqp]
        double* Tm   = Bm + (size_t)MT * nqp;                               // [nq][MT]
        double* xbar = Tm + (size_t)MT * nq;                                // [ns]
        double* cvec = xbar + ns;                                           // [ns]
        double* cred = cvec + ns;                                           // [NW][ns]
        const double* Xb = ep.Xb + b * (size_t)ns * M;
        const int lane = r & 31, warp = r >> 5;
        for (int s = warp; s < ns; s += C::NW) {                            // Eq.9-11
            double acc = 0.0;
            for (int m = lane; m < M; m += 32) acc += Xb[(size_t)s * M + m];
            acc = warp_sum(acc) / (double)M;
            if (lane == 0) xbar[s] = acc;
            for (int m = lane; m < MT; m += 32) Bm[m * nqp + 1 + s] = (m < M) ? Xb[(size_t)s * M + m] - acc : 0.0;
        }
        if (r < MT) {
            Bm[r * nqp] = (r < M) ? ep.g[b * M + r] : 0.0;
            if (nqp > nq) Bm[r * nqp + nq] = 0.0;
        }
        const double lamk = (r < M) ? ep.lam[b * M + inv[r]] : 1.0;
        __syncthreads();
        const double tk_scale = (r < M) ? 1.0 / lamk : 0.0;
        const double sk = (r < M) ? sqrt((double)(M - 1)) * rsqrt(lamk) : 0.0;
        double tk = 0.0;
        const double2* Bm2 = reinterpret_cast<const double2*>(Bm);
        const int nqh = nqp >> 1;
        for (int q = 0; q < nqp; q += 2) {                                  // two right-hand sides per pass over z
            double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
            const double2* bq = Bm2 + (q >> 1);
#pragma unroll
            for (int c = 0; c + 1 < MT; c += 2) {
                const double2 t0 = bq[c * nqh], t1 = bq[(c + 1) * nqh];
                a0 = fma(z[c], t0.x, a0);     b0 = fma(z[c], t0.y, b0);
                a1 = fma(z[c + 1], t1.x, a1); b1 = fma(z[c + 1], t1.y, b1);
            }
            const double raw[2] = {a0 + a1, b0 + b1};
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int qq = q + u;
                if (qq == 0) {
                    tk = raw[u] * tk_scale;
                    if (r < MT) Tm[r] = tk;                                 // t'_k
                } else if (qq < nq) {
                    if (r < MT) Tm[qq * MT + r] = raw[u] * sk;              // U'[s][k]
                    const double part = warp_sum((r < M) ? raw[u] * tk : 0.0);   // c_s, this warp's share
                    if (lane == 0) cred[warp * ns + (qq - 1)] = part;
                }
            }
        }
        __syncthreads();
        if (r < ns) {
            double c = 0.0;
#pragma unroll
            for (int w = 0; w < C::NW; ++w) c += cred[w * ns + r];
            cvec[r] = c;
        }
        transpose_regs<MT>(z, areg);                                        // (its barriers publish Tm, cvec)
        if (r < M) {
            double* Xa = ep.Xa + b * (size_t)ns * M;
            if (ep.wbar) {
                double a0 = 0.0, a1 = 0.0;
                const double2* t2 = reinterpret_cast<const double2*>(Tm);
#pragma unroll
                for (int k = 0; k < MT; k += 2) {
                    const double2 t = t2[k >> 1];
                    a0 = fma(z[k], t.x, a0);
                    if (k + 1 < MT) a1 = fma(z[k + 1], t.y, a1);
                }
                ep.wbar[b * M + r] = a0 + a1;
            }
            for (int s = 0; s < ns; ++s) {
                double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
                const double2* u2 = reinterpret_cast<const double2*>(Tm + (1 + s) * MT);
#pragma unroll
                for (int k = 0; k < MT; k += 4) {
                    const double2 t = u2[k >> 1], u = u2[(k >> 1) + 1];
                    a0 = fma(z[k], t.x, a0);     a1 = fma(z[k + 1], t.y, a1);
                    a2 = fma(z[k + 2], u.x, a2); a3 = fma(z[k + 3], u.y, a3);
                }
                Xa[(size_t)s * M + r] = xbar[s] + cvec[s] + ((a0 + a1) + (a2 + a3));
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// a5 of letkf_syev_batched_f32 (the paper's precision): the
// reflectors, the replay and the back-transform are fp32, the tridiagonal eigenproblem stays fp64
// (ql_log_kernel / bisect_classify_kernel on the (d, e) the fp32 reduction left, twisted
// factorisations in fp64: the orthogonality of Z to 2e-13 costs nothing next to the 2 M^3 fp32
// flops behind it).  Same three routes as fast_apply; w is written as float on the way.
template <int MT>
__global__ void __launch_bounds__(FastCfg<MT>::NT, (MT == 64) ? 6 : (MT == 48 ? LETKF_AP48 : 16))
fast_apply_f32(float* __restrict__ V_, double* __restrict__ w_, float* __restrict__ wf_, int* __restrict__ info_,
               Workspace ws, int M)
{
    using C = FastCfg<MT>;
    extern __shared__ __align__(16) double sm[];
    double*   areg = sm;                                   // A region (ap_a_doubles)
    float*    aregf = reinterpret_cast<float*>(sm);
    double2*  cs   = reinterpret_cast<double2*>(sm);       // [2][AP_S][MT] while rotating
    float*    Rf   = reinterpret_cast<float*>(sm + ap_a_doubles<MT>());   // reflectors, RefLayout order
    float*    taus = Rf + RefLayout<MT>::TOTAL;
    uint32_t* hdr  = reinterpret_cast<uint32_t*>(Rf + ((refl_doubles<MT>() + 3) & ~3));
    int*      inv  = reinterpret_cast<int*>(hdr + ap_hdr_words<MT>(ws.swcap));
    const int r = threadIdx.x;
    const size_t b = blockIdx.x;
    const int flag = ws.flags[b];
    const bool direct = flag == FLAG_GETVEC;
    bool flagged = flag == FLAG_SLOW;
    const int nsw = (flag == FLAG_REPLAY) ? ws.nsweeps[b] : 0;
    const double2* rot = ws.rot + b * ws.logcap;
    constexpr int HT = MT < 32 ? MT : 32;
    for (int s = r; s < nsw; s += C::NT) hdr[s] = ws.hdr[b * ws.swcap + s];
    if (!flagged && r < M) inv[ws.perm[b * M + r]] = r;
    {
        const float* src = reinterpret_cast<const float*>(ws.refl + b * ws.reflstride);
        for (int k = 4 * r; k < refl_doubles<MT>(); k += 4 * C::NT) cp_async16(Rf + k, src + k);
    }
    float z[MT];
    bool columns = false;
    if (direct) {
        double zd[MT];
        const bool ok = direct_eigenvectors<MT>(zd, hdr, areg, ws, w_, b, M, inv);
        __syncthreads();
        if (ok) {
            columns = true;
#pragma unroll
            for (int c = 0; c < MT; ++c) z[c] = (float)zd[c];
        } else {
            flagged = true;
        }
    } else if (!flagged) {
#pragma unroll
        for (int c = 0; c < MT; ++c) z[c] = (c == r) ? 1.0f : 0.0f;
        __syncthreads();
        int spos = 0;
        auto stage = [&](int round) {
            double2* dst = cs + (round & 1) * AP_S * MT;
#pragma unroll
            for (int t = 0; t < AP_S; ++t) {
                const int s = round * AP_S + t;
                if (s < nsw) {
                    const uint32_t h = hdr[s];
                    const int lo = h & 0xffff, m = h >> 16;
                    if (r < MT) {
                        if (r >= lo && r < m) cp_async16(dst + t * MT + r, rot + spos + (m - 1 - r));
                        else dst[t * MT + r] = make_double2(1.0, 0.0);
                    }
                    spos += m - lo;
                }
            }
        };
        const int nrounds = (nsw + AP_S - 1) / AP_S;
        if (nrounds > 0) stage(0);
        cp_async_wait_all();
        __syncthreads();
        for (int k = 0; k < nrounds; ++k) {
            if (k + 1 < nrounds) stage(k + 1);
            const double2* cur = cs + (k & 1) * AP_S * MT;
            const int send = min(nsw, (k + 1) * AP_S);
#pragma unroll 1
            for (int s = k * AP_S; s < send; ++s) {
                const uint32_t h = hdr[s];
                apply_sweep<MT>(z, cur + (s - k * AP_S) * MT, h & 0xffff, h >> 16);
            }
            cp_async_wait_all();
            __syncthreads();
        }
    }
    if (flagged) {
        double*  dsm  = areg;
        double*  esm  = areg + MT;
        double2* sink = reinterpret_cast<double2*>(areg + 2 * MT);
        double2* csb  = sink + MT;
        int*     ctl  = reinterpret_cast<int*>(csb + MT);
        __syncthreads();
#pragma unroll
        for (int c = 0; c < MT; ++c) z[c] = (c == r) ? 1.0f : 0.0f;
        if (r < M) { dsm[r] = ws.dws[b * M + r]; esm[r] = ws.ews[b * M + r]; }
        __syncthreads();
        QLState st{0, 0, 0, 0.0};
        if (r == 0) { esm[M - 1] = 0.0; st.thr = ql_threshold(dsm, esm, 1, M); }
        for (;;) {
            if (r == 0) {
                int lo = 0, m = 0;
                ctl[0] = ql_next_sweep(st, dsm, esm, 1, M, sink, M, lo, m);
                ctl[1] = lo; ctl[2] = m;
            }
            __syncthreads();
            if (ctl[0] != 1) break;
            const int lo = ctl[1], m = ctl[2];
            if (r < MT) csb[r] = (r >= lo && r < m) ? sink[m - 1 - r] : make_double2(1.0, 0.0);
            __syncthreads();
            apply_sweep<MT>(z, csb, lo, m);
            __syncthreads();
        }
        int* permsm = reinterpret_cast<int*>(sink);
        if (r == 0) { sort_eigenvalues(dsm, 1, permsm, 1, M); ctl[3] = st.fail; }
        __syncthreads();
        if (r < M) { inv[permsm[r]] = r; w_[b * M + r] = dsm[r]; }
        if (r == 0 && info_) info_[b] = ctl[3] | 0x40000000;
        __syncthreads();
    }
    cp_async_wait_all();
    __syncthreads();
    if (r < M) wf_[b * M + r] = (float)w_[b * M + r];
    if (!columns) transpose_regs<MT>(z, aregf);
    q_groups_up<MT, 0, (MT - 2) / 8>(z, static_cast<const float*>(Rf), static_cast<const float*>(taus), M, 0);
    // sorted, row-major V through the tile, HT rows per pass
    float* V = V_ + b * M * M;
    float* tile = aregf;
    const int oc = (r < M) ? inv[r] : 0;
#pragma unroll
    for (int r0 = 0; r0 < MT; r0 += HT) {
        if (r0 < M) {
            __syncthreads();
            if (r < M) {
#pragma unroll
                for (int rr = 0; rr < HT; ++rr)
                    if (r0 + rr < MT) tile[rr * C::LDT + oc] = z[r0 + rr];
            }
            __syncthreads();
            if (r < M) {
                const int nr = min(HT, M - r0);
#pragma unroll 8
                for (int rr = 0; rr < nr; ++rr) V[(size_t)(r0 + rr) * M + r] = tile[rr * C::LDT + r];
            }
        }
    }
}
template <int MT> size_t fast_apply_f32_smem(int swcap)
{
    return sizeof(double) * (size_t)ap_a_doubles<MT>() + sizeof(float) * (size_t)((refl_doubles<MT>() + 3) & ~3)
         + sizeof(uint32_t) * (size_t)ap_hdr_words<MT>(swcap) + sizeof(int) * MT + 16;
}

// M = 1 of the fp32 entry point
__global__ void f32_order_one(const float* __restrict__ A, float* __restrict__ w, float* __restrict__ V, int* __restrict__ info, int batch)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < batch) { w[b] = A[b]; V[b] = 1.0f; if (info) info[b] = 0; }
}

static inline bool fast_supported(int M) { return M >= 2 && M <= 64; }
static inline int fast_bucket(int M) { return M <= 16 ? 16 : (M <= 32 ? 32 : (M <= 48 ? 48 : 64)); }
static inline int fast_refl_doubles(int M)
{
    switch (fast_bucket(M)) {
        case 16: return refl_doubles<16>();
        case 32: return refl_doubles<32>();
        case 48: return refl_doubles<48>();
        default: return refl_doubles<64>();
    }
}

}  // namespace letkf

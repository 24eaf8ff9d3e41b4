// common.cuh -- shared device helpers of libletkf (CUDA path only; the CPU oracle shares nothing
// with this tree).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace letkf {

// Per-matrix workspace layout (device).  One record per matrix of the current chunk.
//   dws, ews  : the tridiagonal form T = Q^T A Q (kept untouched after the reduction so the
//               slow path can restart from it)
//   perm      : perm[k] = index (in QL order) of the k-th smallest eigenvalue
//   hdr       : one word per QL sweep, lo | (m << 16): rotations i = m-1 ... lo
//   rot       : (c, s) of every rotation, in application order
struct Workspace {
    double*   dws;      // [chunk][M]
    double*   ews;      // [chunk][M]
    int*      perm;     // [chunk][M]
    int*      nsweeps;  // [chunk]
    int*      flags;    // [chunk]   FLAG_REPLAY: replay the log; FLAG_SLOW: log unusable, classic iteration in the apply
                        //           kernel; FLAG_GETVEC: no log, eigenvectors by twisted factorisation
    uint32_t* hdr;      // [chunk][swcap]
    double2*  rot;      // [chunk][logcap]
    double*   refl;     // [chunk][reflstride]  M <= 64: the Householder reflectors and their taus (RefLayout)
    double*   s1;       // [chunk][M]  eigenvalues of the first QL pass by position (classify mode; else unused)
    int       swcap;
    int       logcap;
    int       reflstride;
    unsigned long long* rot_counter;   // profiling only (NULL otherwise): total rotations logged
};

__host__ __device__ inline int sweep_capacity(int M) { return 6 * M + 32; }
// rotations the log of one matrix holds.  One-pass QL (Wilkinson shifts): measured mean 1.05 M^2, max
// 1.36 M^2 over the configured workloads -> 2 M^2.  Two-pass QL (second pass shifted by the
// eigenvalues of the first): mean 0.71 M^2, max 0.81 M^2 -> M^2.  A matrix that needs more is
// finished by the slow path (flags[b]).
__host__ __device__ inline int log_capacity(int M, bool two_pass = false)
{
    return (two_pass ? 1 : 2) * M * M + 4 * M + 16;
}

// ---- eigenvectors of T without rotations (fast_apply, M <= 64) -----------------
// A matrix is "easy" when, inside every unreduced block of T, no two eigenvalues are closer than
// GV_TINY ||T|| and no more than GV_PH eigenvalues lie within GV_GAP ||T|| above any eigenvalue: its
// eigenvectors then come from twisted factorisations of T - lambda I (one per thread), and the pairs
// closer than GV_GAP ||T|| are made orthogonal by a first-order symmetric correction.  Every other
// matrix has its rotations logged and replayed.  ql_log_kernel (mode 2) classifies, fast_apply
// follows the flag.
constexpr double GV_GAP  = 4.0e-3;    // eps C / GV_GAP bounds the loss of orthogonality left uncorrected (C ~ 7 measured)
constexpr double GV_TINY = 1.0e-8;    // the correction is first order: (eps C / GV_TINY)^2 must stay far below the tolerance
constexpr int    GV_PH   = 12;        // partners a vector may have on either side (<= 12: the partner lists are three words of
                                      // 8-bit fields).  4 left 29% of config 5's M = 48 matrices (p = 49: the small eigenvalues
                                      // of Yb^T R Yb crowd above the shift) to the logging pass, 6 none; M = 96 with p = 98 has
                                      // up to 10 in the window.  The first-order correction's error grows with the partner
                                      // count: <= 24 (eps C / GV_TINY)^2 ~ 1.4e-13
// Both tests are taken among the eigenvalues of ONE unreduced block of T (the eigenvalue found at position k belongs to the
// block of k): vectors of different blocks have disjoint supports, and a 1 x 1 block's vector is a unit vector.
// partner list of one eigenvector: up to 24 positions (< 256), three words of 8-bit fields, selected without indexing
struct PartnerList {
    unsigned long long w0 = 0ull, w1 = 0ull, w2 = 0ull;
    int np = 0;
    __device__ __forceinline__ void add(int q)
    {
        const unsigned long long v = (unsigned long long)q << (8 * (np & 7));
        if (np < 8) w0 |= v; else if (np < 16) w1 |= v; else if (np < 24) w2 |= v;
        if (np < 24) ++np;
    }
    __device__ __forceinline__ int get(int t) const
    {
        const unsigned long long w = t < 8 ? w0 : (t < 16 ? w1 : w2);
        return (int)((w >> (8 * (t & 7))) & 255ull);
    }
};
// The sorted eigenvalue s (value lam, block id blk > 0, or < 0 for a 1 x 1 block) against the ones above it: returns true
// when the matrix has to go to the rotation log.  val(s), blkid(s) read the sorted sequence.
template <class FV, class FB>
__device__ __forceinline__ bool gv_hard_at(int s, int M, double nrm, FV val, FB blkid)
{
    const int blk = blkid(s);
    if (blk < 0) return false;
    const double lam = val(s);
    int cnt = 0;
    for (int u = s + 1; u < M; ++u) {
        const double gap = val(u) - lam;
        if (!(gap < GV_GAP * nrm)) break;
        if (blkid(u) != blk) continue;
        if (gap < GV_TINY * nrm) return true;
        if (++cnt > GV_PH) return true;
    }
    return false;
}
// Splitting T (reading G24): an off-diagonal |e_i| <= GV_SPLIT 2^-53 ||T|| (or 2^-53 (|d_i| + |d_i+1|)) is set to exactly 0
// before any solver sees the matrix -- a backward error of GV_SPLIT eps ||T|| per entry, 2 sqrt(2 M) eps ||T|| in all.  The
// factor is what the rounding of the reduction leaves in the part of T that belongs to a repeated eigenvalue (measured on
// config 5, M = 128 ... 256 with p = 98: 1e-17 ... 6e-16 ||T||): with it such a cluster falls apart into 1 x 1 blocks.
constexpr double GV_SPLIT = 8.0;
constexpr int    FLAG_REPLAY = 0, FLAG_SLOW = 1, FLAG_GETVEC = 2, FLAG_PENDING = 3;   // Workspace::flags (PENDING: between
                                                                                     // the classifying and the logging QL kernel)

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Deterministic block-wide sum; red must hold NT/32 doubles.  All threads get the result.
template <int NT>
__device__ __forceinline__ double block_sum(double v, double* red)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    v = warp_sum(v);
    if (lane == 0) red[warp] = v;
    __syncthreads();
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < NT / 32; ++w) t += red[w];
    __syncthreads();
    return t;
}

// ---------------------------------------------------------------------------------------------
// Implicit-shift QL on a symmetric tridiagonal matrix ("The eigenvalues and
// eigenvectors of the tridiagonal matrix are computed by the implicit QL method as in
// EISPACK/LAPACK").  Only the scalar recurrences are run here; every plane rotation (c, s) is
// written to `sink` and applied to the eigenvector matrix elsewhere, so the serial chain
// (sqrt/div latency) never stalls the threads that own the matrix.
//
// d[i*stride], e[i*stride]: diagonal / off-diagonal (e[i] couples i and i+1; e[M-1] unused).
// One call produces the next non-empty sweep: rotations for i = m-1 ... lo, stored at
// sink[0 .. m-lo-1], to be applied as
//      f = z[i+1];  z[i+1] = s*z[i] + c*f;  z[i] = c*z[i] - s*f      (columns of Z).
// Returns 1 with (lo, m) set, 0 when all eigenvalues have converged, -1 if the sweep would not
// fit into sink_cap (nothing is changed in that case).
// Conventions fixed in DESIGN.md reading G10: Wilkinson shift, deflation when
// |e_m| <= 2^-53 max(|d_m| + |d_m+1|, max_i(|d_i| + |e_i|)), at most QL_MAX_SWEEPS sweeps per eigenvalue
// (then st.fail is bumped).
struct QLState { int l; int iter; int fail; double thr; };   // thr = 2^-53 max_i(|d_i| + |e_i|), set by ql_threshold

constexpr int QL_MAX_SWEEPS = 60;    // per eigenvalue (reading G10)

// Deflation threshold relative to the whole matrix (EISPACK tql2's running norm, taken once):
// |e_m| <= 2^-53 max(|d_m| + |d_m+1|, max_i(|d_i| + |e_i|)).  The purely local test of LAPACK stalls
// on eigenvalues far below eps ||T|| of a matrix that is not graded (measured: > 30 sweeps).
__device__ __forceinline__ double ql_threshold(const double* d, const double* e, int stride, int M)
{
    double t = 0.0;
    for (int i = 0; i < M; ++i) t = fmax(t, fabs(d[(size_t)i * stride]) + (i < M - 1 ? fabs(e[(size_t)i * stride]) : 0.0));
    return 1.1102230246251565e-16 * t;
}

#define LETKF_LD(i) d[(size_t)(i) * stride]
#define LETKF_LE(i) e[(size_t)(i) * stride]

// Advance past converged eigenvalues; returns true with (l = st.l, m) when the block [l, m] needs
// another sweep, false when everything has converged.
__device__ __forceinline__ bool ql_find_block(QLState& st, const double* d, const double* e, int stride,
                                              int M, int& m_out)
{
    const double eps = 1.1102230246251565e-16;   // 2^-53
    while (st.l < M) {
        const int l = st.l;
        int m = l;
        for (; m < M - 1; ++m) {
            const double dd = fabs(LETKF_LD(m)) + fabs(LETKF_LD(m + 1));
            if (fabs(LETKF_LE(m)) <= fmax(eps * dd, st.thr)) break;
        }
        if (m == l) { st.l = l + 1; st.iter = 0; continue; }
        if (st.iter >= QL_MAX_SWEEPS) { st.fail += 1; st.l = l + 1; st.iter = 0; continue; }
        st.iter += 1;
        m_out = m;
        return true;
    }
    return false;
}

// Wilkinson shift for the block [l, m]: returns the starting value of g.
__device__ __forceinline__ double ql_shift(const double* d, const double* e, int stride, int l, int m)
{
    const double el = LETKF_LE(l);
    double g = (LETKF_LD(l + 1) - LETKF_LD(l)) / (2.0 * el);
    const double r = sqrt(g * g + 1.0);
    return LETKF_LD(m) - LETKF_LD(l) + el / (g + copysign(r, g));
}

// One plane rotation of the sweep (index i).  Returns false if the sweep must stop here
// (underflow / NaN: the block is split at i+1 and no rotation is produced).
__device__ __forceinline__ bool ql_rot_step(double* d, double* e, int stride, int i, int m,
                                            double& s, double& c, double& p, double& g, double2& cs_out)
{
    const double ei = LETKF_LE(i);
    const double f = s * ei;
    const double b = c * ei;
    const double r2 = f * f + g * g;
    if (!(r2 > 0.0)) {
        LETKF_LE(i + 1) = 0.0;
        LETKF_LD(i + 1) -= p;
        LETKF_LE(m) = 0.0;
        return false;
    }
    const double rinv = rsqrt(r2);
    LETKF_LE(i + 1) = r2 * rinv;
    s = f * rinv;
    c = g * rinv;
    g = LETKF_LD(i + 1) - p;
    const double r = (LETKF_LD(i) - g) * s + 2.0 * c * b;
    p = s * r;
    LETKF_LD(i + 1) = g + p;
    g = c * r - b;
    cs_out = make_double2(c, s);
    return true;
}

__device__ __forceinline__ void ql_finish_sweep(double* d, double* e, int stride, int l, int m, double p, double g)
{
    LETKF_LD(l) -= p;
    LETKF_LE(l) = g;
    LETKF_LE(m) = 0.0;
}

// Single-thread form: produces the next non-empty sweep (see the header comment above).
__device__ __forceinline__ int ql_next_sweep(QLState& st, double* d, double* e, int stride, int M,
                                             double2* sink, int sink_cap, int& lo_out, int& m_out)
{
    for (;;) {
        int m;
        if (!ql_find_block(st, d, e, stride, M, m)) return 0;
        const int l = st.l;
        if (m - l > sink_cap) { st.iter -= 1; return -1; }
        double g = ql_shift(d, e, stride, l, m);
        double s = 1.0, c = 1.0, p = 0.0;
        int i;
        for (i = m - 1; i >= l; --i) {
            double2 cs;
            if (!ql_rot_step(d, e, stride, i, m, s, c, p, g, cs)) break;
            sink[m - 1 - i] = cs;
        }
        int lo;
        if (i >= l) lo = i + 1;
        else { ql_finish_sweep(d, e, stride, l, m, p, g); lo = l; }
        if (m - lo > 0) { lo_out = lo; m_out = m; return 1; }
    }
}

// Ascending insertion sort of d with the permutation that sorts it.  The QL iteration tends to
// leave the eigenvalues in roughly descending order (insertion sort's worst case: it was 28% of the
// classifying QL kernel), so a sequence with more descents than ascents is reversed first.
__device__ __forceinline__ void sort_eigenvalues(double* d, int dstride, int* perm, int pstride, int M)
{
    int desc = 0;
    for (int k = 0; k + 1 < M; ++k) desc += d[(size_t)k * dstride] > d[(size_t)(k + 1) * dstride] ? 1 : 0;
    if (2 * desc > M) {
        for (int k = 0; k < M / 2; ++k) {
            const double t = d[(size_t)k * dstride];
            d[(size_t)k * dstride] = d[(size_t)(M - 1 - k) * dstride];
            d[(size_t)(M - 1 - k) * dstride] = t;
        }
        for (int k = 0; k < M; ++k) perm[(size_t)k * pstride] = M - 1 - k;
    } else {
        for (int k = 0; k < M; ++k) perm[(size_t)k * pstride] = k;
    }
    for (int k = 1; k < M; ++k) {
        const double val = d[(size_t)k * dstride];
        const int pk = perm[(size_t)k * pstride];
        int j = k - 1;
        while (j >= 0 && d[(size_t)j * dstride] > val) {
            d[(size_t)(j + 1) * dstride] = d[(size_t)j * dstride];
            perm[(size_t)(j + 1) * pstride] = perm[(size_t)j * pstride];
            --j;
        }
        d[(size_t)(j + 1) * dstride] = val;
        perm[(size_t)(j + 1) * pstride] = pk;
    }
}

#undef LETKF_LD
#undef LETKF_LE

}  // namespace letkf

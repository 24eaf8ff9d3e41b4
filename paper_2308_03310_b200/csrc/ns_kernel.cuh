// ns_kernel.cuh -- the EVD-FREE form of the local analysis (the paper's stated
// future work: "explore algorithms that can avoid divergence").
//
// Eq.14-16 need only two functions of Q = ((M-1)/rho) I + dY^T R dY (Eq.17):  Pa = Q^-1 (applied to a
// vector) and Pa^1/2 = Q^-1/2.  Both come out of the coupled Newton-Schulz iteration for the matrix
// square root (Higham, Functions of Matrices, Eq.6.35) without any eigendecomposition:
//     B = Q / c,  Y_0 = B,  Z_0 = I;   T_k = (3 I - Z_k Y_k) / 2,  Y_k+1 = Y_k T_k,  Z_k+1 = Z_k T_k
//     Y_k -> B^1/2,  Z_k -> B^-1/2            (quadratically once ||I - Z Y|| < 1; all iterates are
//                                              polynomials in B: symmetric, and they commute)
// so  Q^-1/2 = Z / sqrt(c),  W = sqrt(M-1) Q^-1/2  (the symmetric principal root, reading G2),
// wbar = Q^-1 g = Z (Z g) / c.  Three M x M x M products per iteration and nothing else: the one
// formulation of the path that is a dense contraction throughout, so it runs on the FP64 tensor
// cores (mma.sync.m8n8k4.f64), with no data-dependent branch but the convergence test.
// Scaling: lambda_min(Q) >= (M-1)/rho (the low-rank part is positive semi-definite) and
// lambda_max(Q) <= ||Q||_inf =: u; with c = u / 1.5 the spectrum of B lies in
// (0, 1.5], inside the iteration's region of convergence (0, 3).  The iteration count grows like
// log_1.5 sqrt(kappa(Q)): 6 at kappa = 4 (config 4), 11 at kappa = 300 -- 36 to 66 M^3 flops against
// the ~5.4 M^3 of the EVD route, which is why this form loses on B200, where the fp64 tensor rate
// equals the vector rate (measured: DESIGN.md section 5); it is kept as the divergence-free
// alternative and as an independent route to the same numbers.
// Accuracy (measured against the oracle): the coupled iteration is not backward stable -- Y_k = B Z_k
// only holds up to the rounding errors committed so far, which later steps do not repair -- and W, Xa
// come out within ~3e-14 kappa(Q)^2 of the EVD route's: 1e-12 at config 4 (kappa ~ 4), 3e-9 at
// kappa ~ 300, 2e-7 at kappa ~ 3e3.  (A final step Z <- Z (3I - Z B Z)/2 against the original B, the
// uncoupled Newton-Schulz step, makes it worse: that iteration is unstable for kappa >> 1; tried.)
#pragma once
#include "common.cuh"

namespace letkf {

constexpr int NS_MT = 64;          // padded order (the register-path sizes, M <= 64)
constexpr int NS_LD = 68;          // row stride: fragments of both operands are conflict-free per half warp
constexpr int NS_NT = 128;         // 4 warps, each owns a 16-row strip of every product
constexpr int NS_MAXIT = 40;
constexpr size_t NS_SMEM = sizeof(double) * (3 * (size_t)NS_MT * NS_LD + 4 * NS_MT + 16 * NS_MT + 32);

__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// acc (16 x 64 strip of rows 16w ..) = A[strip rows][:] * B, both 64 x 64 in shared memory (stride NS_LD).
// Fragments (PTX m8n8k4): A: lane l holds A[l/4][l%4]; B: lane l holds B[l%4][l/4];
// C: lane l holds C[l/4][2(l%4)], C[l/4][2(l%4)+1].
__device__ __forceinline__ void strip_gemm(double (&acc)[2][8][2], const double* A, const double* B, int warp, int lane)
{
#pragma unroll
    for (int t = 0; t < 2; ++t)
#pragma unroll
        for (int ct = 0; ct < 8; ++ct) { acc[t][ct][0] = 0.0; acc[t][ct][1] = 0.0; }
    const double* arow0 = A + (16 * warp + (lane >> 2)) * NS_LD + (lane & 3);
    const double* brow = B + (lane & 3) * NS_LD + (lane >> 2);
#pragma unroll 4
    for (int kk = 0; kk < NS_MT / 4; ++kk) {
        const double a0 = arow0[4 * kk], a1 = arow0[8 * NS_LD + 4 * kk];
        const double* bk = brow + 4 * kk * NS_LD;
#pragma unroll
        for (int ct = 0; ct < 8; ++ct) {
            const double bv = bk[8 * ct];
            dmma884(acc[0][ct], a0, bv);
            dmma884(acc[1][ct], a1, bv);
        }
    }
}

__device__ __forceinline__ void strip_store(double* C, const double (&acc)[2][8][2], int warp, int lane)
{
#pragma unroll
    for (int t = 0; t < 2; ++t)
#pragma unroll
        for (int ct = 0; ct < 8; ++ct)
            *reinterpret_cast<double2*>(C + (16 * warp + 8 * t + (lane >> 2)) * NS_LD + 8 * ct + 2 * (lane & 3)) =
                make_double2(acc[t][ct][0], acc[t][ct][1]);
}

// One CTA per grid point.  info[b] = number of iterations taken, or 0x20000000 | iterations if the
// residual ||I - Z Y||_F did not reach the tolerance within NS_MAXIT (result then not to be trusted).
__global__ void __launch_bounds__(NS_NT)
ns_analysis_kernel(const double* __restrict__ Yb_, const double* __restrict__ d_, const double* __restrict__ r_,
                   const double* Xb_, int M, int p, int ns, double rho,
                   double* Xa_, double* __restrict__ W_, double* __restrict__ wbar_, int* __restrict__ info)
{
    extern __shared__ __align__(16) double sm[];
    double* Ys = sm;                               // [64][68]
    double* Zs = Ys + NS_MT * NS_LD;
    double* Ts = Zs + NS_MT * NS_LD;               // also the staging area of the observations
    double* gs = Ts + NS_MT * NS_LD;               // [64] g = dY^T (r o d)
    double* v1 = gs + NS_MT;                       // [64]
    double* wb = v1 + NS_MT;                       // [64] wbar
    double* red = wb + NS_MT;                      // [64] reductions
    double* dX = red + NS_MT;                      // [ns <= 16][64]
    double* xbar = dX + 16 * NS_MT;                // [16]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const size_t b = blockIdx.x;
    const double* Yb = Yb_ + b * (size_t)p * M;
    const double* dv = d_ + b * (size_t)p;
    const double* rv = r_ + b * (size_t)p;
    const double shift = (double)(M - 1) / rho;

    // ---- a1, a2: Q (rows m = tid / 2, columns 32 (tid % 2) ...) and g, observations staged 16 rows at a time
    const int m = tid >> 1, n0 = 32 * (tid & 1);
    double acc1[32];
#pragma unroll
    for (int c = 0; c < 32; ++c) acc1[c] = 0.0;
    double gm = 0.0, tr = 0.0;
    double* stage = Ts;                            // [16][64] rows, then r, r d
    for (int j0 = 0; j0 < p; j0 += 16) {
        const int nj = min(16, p - j0);
        __syncthreads();
        for (int idx = tid; idx < 16 * NS_MT; idx += NS_NT) {
            const int jj = idx >> 6, cc = idx & 63;
            stage[idx] = (jj < nj && cc < M) ? Yb[(size_t)(j0 + jj) * M + cc] : 0.0;
        }
        if (tid < 16) { stage[16 * NS_MT + tid] = tid < nj ? rv[j0 + tid] : 0.0; stage[17 * NS_MT + tid] = tid < nj ? rv[j0 + tid] * dv[j0 + tid] : 0.0; }
        __syncthreads();
        for (int jj = 0; jj < nj; ++jj) {
            const double* y = stage + jj * NS_MT;
            const double rj = stage[16 * NS_MT + jj];
            const double ym = y[m], rym = rj * ym;
            if ((tid & 1) == 0) { gm = fma(ym, stage[17 * NS_MT + jj], gm); tr = fma(rym, ym, tr); }
            const double2* y2 = reinterpret_cast<const double2*>(y + n0);
#pragma unroll
            for (int c = 0; c < 16; ++c) {
                const double2 t = y2[c];
                acc1[2 * c] = fma(rym, t.x, acc1[2 * c]);
                acc1[2 * c + 1] = fma(rym, t.y, acc1[2 * c + 1]);
            }
        }
    }
    __syncthreads();
    // ||Q||_inf (largest absolute row sum) >= lambda_max -> scaling
    {
        double rs = 0.0;
#pragma unroll
        for (int cc = 0; cc < 32; ++cc) {
            const int n = n0 + cc;
            if (m < M && n < M) rs += fabs(acc1[cc] + ((m == n) ? shift : 0.0));
        }
        rs += __shfl_xor_sync(0xffffffffu, rs, 1);              // the two halves of row m sit in neighbouring lanes
        if ((tid & 1) == 0) { red[m] = rs; gs[m] = (m < M) ? gm : 0.0; }
    }
    (void)tr;
    __syncthreads();
    double u = shift;
    for (int i = 0; i < NS_MT; ++i) u = fmax(u, red[i]);
    const double c = u / 1.5, cinv = 1.0 / c;
    // Y_0 = Q / c (padded rows / columns: identity block scaled like the shift, harmless), Z_0 = I
#pragma unroll
    for (int cc = 0; cc < 32; ++cc) {
        const int n = n0 + cc;
        double q = acc1[cc] + ((m == n) ? shift : 0.0);
        if (m >= M || n >= M) q = (m == n) ? shift : 0.0;
        Ys[m * NS_LD + n] = q * cinv;
        Zs[m * NS_LD + n] = (m == n) ? 1.0 : 0.0;
    }
    // ensemble statistics (Eq.9-11) meanwhile
    const double* Xb = Xb_ + b * (size_t)ns * M;
    for (int s = warp; s < ns; s += NS_NT / 32) {
        double a = 0.0;
        for (int k = lane; k < M; k += 32) a += Xb[(size_t)s * M + k];
        a = warp_sum(a) / (double)M;
        if (lane == 0) xbar[s] = a;
        for (int k = lane; k < NS_MT; k += 32) dX[s * NS_MT + k] = (k < M) ? Xb[(size_t)s * M + k] - a : 0.0;
    }
    __syncthreads();

    // ---- coupled Newton-Schulz on the FP64 tensor cores
    double accm[2][8][2];
    int it = 0;
    bool conv = false;
    double r2prev = 1.0;
    const double tol2 = 1e-28 * (double)M;                      // ||I - Z Y||_F <= 1e-14 sqrt(M)
    for (; it < NS_MAXIT; ++it) {
        strip_gemm(accm, Zs, Ys, warp, lane);                   // P = Z Y
        double res = 0.0;
#pragma unroll
        for (int t = 0; t < 2; ++t)
#pragma unroll
            for (int ct = 0; ct < 8; ++ct) {
                const int row = 16 * warp + 8 * t + (lane >> 2), col = 8 * ct + 2 * (lane & 3);
                const double e0 = ((row == col) ? 1.0 : 0.0) - accm[t][ct][0];
                const double e1 = ((row == col + 1) ? 1.0 : 0.0) - accm[t][ct][1];
                res = fma(e0, e0, fma(e1, e1, res));
                accm[t][ct][0] = ((row == col) ? 1.0 : 0.0) + 0.5 * e0;        // T = (3 I - P) / 2 = I + (I - P) / 2
                accm[t][ct][1] = ((row == col + 1) ? 1.0 : 0.0) + 0.5 * e1;
            }
        strip_store(Ts, accm, warp, lane);
        res = warp_sum(res);
        if (lane == 0) red[warp] = res;
        __syncthreads();                                        // T complete, partial residuals visible
        const double r2 = (red[0] + red[1]) + (red[2] + red[3]);
        // converged: at the tolerance, or at the rounding floor of the iteration (eps kappa^1/2-ish: the
        // residual was already small and has stopped falling quadratically)
        if (r2 <= tol2 || (r2prev <= 1e-12 && r2 >= 1e-3 * r2prev)) { conv = true; break; }
        if (!(r2 == r2)) break;                                 // NaN input: give up
        r2prev = r2;
        strip_gemm(accm, Ys, Ts, warp, lane);                   // Y <- Y T (own rows of Y are the A operand: in place)
        __syncwarp();
        strip_store(Ys, accm, warp, lane);
        strip_gemm(accm, Zs, Ts, warp, lane);                   // Z <- Z T
        __syncwarp();
        strip_store(Zs, accm, warp, lane);
        __syncthreads();                                        // Y, Z complete for the next product; red reusable
    }
    if (tid == 0 && info) info[b] = conv ? it : (0x20000000 | it);

    // ---- a6: wbar = Q^-1 g = Z (Z g) / c ;  a7: W = sqrt(M-1) Z / sqrt(c)
    if (tid < NS_MT) {
        double a = 0.0;
        for (int n = 0; n < NS_MT; ++n) a = fma(Zs[tid * NS_LD + n], gs[n], a);
        v1[tid] = a;
    }
    __syncthreads();
    if (tid < NS_MT) {
        double a = 0.0;
        for (int n = 0; n < NS_MT; ++n) a = fma(Zs[tid * NS_LD + n], v1[n], a);
        a *= cinv;
        wb[tid] = a;
        if (wbar_ && tid < M) wbar_[b * M + tid] = a;
    }
    const double wscale = sqrt((double)(M - 1)) * rsqrt(c);
    if (W_) {
        double* Wo = W_ + b * (size_t)M * M;
        for (int idx = tid; idx < M * M; idx += NS_NT) {
            const int rr = idx / M, cc = idx - rr * M;
            Wo[idx] = wscale * Zs[rr * NS_LD + cc];
        }
    }
    __syncthreads();
    // ---- a9: Xa[s][mm] = xbar_s + dX_s . wbar + sum_k dX[s][k] W[k][mm]
    double* Xa = Xa_ + b * (size_t)ns * M;
    for (int idx = tid; idx < ns * NS_MT; idx += NS_NT) {
        const int s = idx >> 6, mm = idx & 63;
        if (mm >= M) continue;
        double a0 = 0.0, a1 = 0.0;
        for (int k = 0; k < M; ++k) {
            const double dx = dX[s * NS_MT + k];
            a0 = fma(dx, wb[k], a0);
            a1 = fma(dx, Zs[k * NS_LD + mm], a1);
        }
        Xa[(size_t)s * M + mm] = xbar[s] + a0 + wscale * a1;
    }
}

}  // namespace letkf

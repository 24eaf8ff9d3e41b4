// big_kernels.cuh -- M > 64: the eigenvectors without rotations (step a5 as a dense contraction).
//
// Above the register path the apply step was a replay of ~0.7 M^2 logged plane rotations on the rows of
// Q^T (mid_apply / generic_apply: 4.4 M^3 flops, chain-latency or HBM bound, 45-60% of the step).
// The route of fast_apply carries over: where the classifier of ql_log_kernel (common.cuh, GV_*) finds
// the spectrum separated well enough, the eigenvectors of T come from twisted factorisations of
// T - lambda I (big_getvec: one thread per eigenvector, the vector in global memory / L2 instead of
// registers, Z[i][k] so that the threads of a warp touch consecutive words), and
//     V = Q Z,   i.e.  V^T = Z^T (Q^T)
// is one M x M x M product on the FP64 tensor cores (big_gemm, mma.sync.m8n8k4.f64) -- 2 M^3 flops
// at the DMMA rate instead of 4.4 M^3 at a fraction of the DFMA rate.  Matrices the classifier
// leaves to the rotation log (FLAG_REPLAY) or to the classic iteration (FLAG_SLOW) keep the kernels
// of mid_kernels.cuh / generic_kernels.cuh, which skip the matrices finished here.
//
// Z lives in the matrix's record of the rotation log, which this route never writes: logcap double2
// = 2 (M^2 + 4 M + 16) doubles: Z in the first M^2, the staging of V for M > 128 in the second.
#pragma once
#include "common.cuh"
#include "fast_kernels.cuh"
#include "ns_kernel.cuh"

namespace letkf {

constexpr int BIG_NT = 256;
static inline size_t big_getvec_smem(int M)
{
    // ds, es, wsrt; perm, inv; the tile of the correction [8][M] and its coefficients [2 GV_PH][ceil32(M)]
    return sizeof(double) * (3 * (size_t)M + 8 * (size_t)M + 2 * GV_PH * (size_t)((M + 31) / 32 * 32)) + sizeof(int) * 4 * (size_t)M + 64;
}

__device__ __forceinline__ double* big_z(const Workspace& ws, size_t b) { return reinterpret_cast<double*>(ws.rot + b * ws.logcap); }

__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gmem_src)
{
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gmem_src) : "memory");
}

// One CTA of ceil32(M) threads per matrix, thread k = position k of T.  The arithmetic is getvec<MT> /
// direct_eigenvectors<MT> of fast_kernels.cuh restricted to the unreduced block [lo, hi] of position
// k, with the vector in Z[.][k].  Every pass that reads the vector back takes it eight entries at a
// time (the loads of a block are independent of the recurrence: one L2 latency per eight steps).
constexpr int BIG_PF = 8;
__global__ void __launch_bounds__(BIG_NT, 2)
big_getvec(Workspace ws, const double* __restrict__ w_, int M)
{
    extern __shared__ __align__(16) double bg_sm[];
    double* ds = bg_sm;                                   // [M]
    double* es = ds + M;                                  // [M] negligible entries exactly 0
    double* wsrt = es + M;                                // [M] eigenvalues ascending
    int* perm = reinterpret_cast<int*>(wsrt + M);         // [M] position of the k-th smallest
    int* inv = perm + M;                                  // [M]
    __shared__ double red[BIG_NT / 32];
    const size_t b = blockIdx.x;
    if (ws.flags[b] != FLAG_GETVEC) return;
    const int k = threadIdx.x, nwarps = blockDim.x >> 5;
    double* Z = big_z(ws, b);
    const double eps = 1.1102230246251565e-16;

    double nrm = 0.0;
    if (k < M) {
        const double dk = ws.dws[b * M + k], ek = (k < M - 1) ? ws.ews[b * M + k] : 0.0;
        ds[k] = dk; es[k] = ek;
        wsrt[k] = w_[b * M + k];
        perm[k] = ws.perm[b * M + k];
        nrm = fabs(dk) + fabs(ek);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nrm = fmax(nrm, __shfl_xor_sync(0xffffffffu, nrm, o));
    if ((k & 31) == 0) red[k >> 5] = nrm;
    __syncthreads();
    nrm = 0.0;
    for (int wq = 0; wq < nwarps; ++wq) nrm = fmax(nrm, red[wq]);
    const double thr = eps * nrm;
    if (k < M) inv[perm[k]] = k;
    bool cut = true;
    if (k < M - 1) cut = fabs(es[k]) <= fmax(eps * (fabs(ds[k]) + fabs(ds[k + 1])), GV_SPLIT * thr);
    __syncthreads();
    if (k < M && cut) es[k] = 0.0;
    __syncthreads();
    int lo = k, hi = k;
    double lam = 0.0;
    if (k < M) {
        while (lo > 0 && es[lo - 1] != 0.0) --lo;
        while (hi < M - 1 && es[hi] != 0.0) ++hi;
        lam = wsrt[inv[k]];
    }
    const bool own = k < M && lo < hi;
    const double pivmin = fmax(thr * eps, 1e-300);
    double res = 0.0;
    if (own) {
        double* zk = Z + k;
        // forward pivots: 1 / D+_i
        {
            double P = ds[lo] - lam;
            for (int i = lo; i <= hi; ++i) {
                P = (fabs(P) < pivmin) ? -pivmin : P;
                const double rp = fast_rcp(P);
                zk[(size_t)i * M] = rp;
                if (i < hi) { const double ei = es[i]; P = fma(-(ei * ei), rp, ds[i + 1] - lam); }
            }
        }
        // backward pivots on the fly: the twist index
        int r = lo;
        {
            double best = 1.7976931348623157e308;
            double Dm = ds[hi] - lam;
            for (int i0 = hi; i0 >= lo; i0 -= BIG_PF) {
                double buf[BIG_PF];
#pragma unroll
                for (int u = 0; u < BIG_PF; ++u) buf[u] = (i0 - u > lo) ? zk[(size_t)(i0 - u - 1) * M] : 0.0;
#pragma unroll
                for (int u = 0; u < BIG_PF; ++u) {
                    const int i = i0 - u;
                    if (i >= lo) {
                        Dm = (fabs(Dm) < pivmin) ? -pivmin : Dm;
                        const double di = ds[i] - lam;
                        double Pi = di;
                        if (i > lo) { const double el = es[i - 1]; Pi = fma(-(el * el), buf[u], di); }
                        Pi = (fabs(Pi) < pivmin) ? -pivmin : Pi;
                        const double gam = fabs(Pi + Dm - di);
                        if (gam < best) { best = gam; r = i; }
                        if (i > lo) { const double el = es[i - 1]; Dm = fma(-(el * el), fast_rcp(Dm), ds[i - 1] - lam); }
                    }
                }
            }
        }
        // from the bottom down to the twist: 1 / D-_i (i > r); below the twist the vector itself
        {
            double Dm = ds[hi] - lam;
            for (int i = hi; i > r; --i) {
                Dm = (fabs(Dm) < pivmin) ? -pivmin : Dm;
                const double rd = fast_rcp(Dm);
                zk[(size_t)i * M] = rd;
                const double el = es[i - 1];              // (i > r >= lo)
                Dm = fma(-(el * el), rd, ds[i - 1] - lam);
            }
            zk[(size_t)r * M] = 1.0;
            double zc = 1.0;
            for (int i0 = r - 1; i0 >= lo; i0 -= BIG_PF) {
                double buf[BIG_PF];
#pragma unroll
                for (int u = 0; u < BIG_PF; ++u) buf[u] = (i0 - u >= lo) ? zk[(size_t)(i0 - u) * M] : 0.0;
#pragma unroll
                for (int u = 0; u < BIG_PF; ++u) {
                    const int i = i0 - u;
                    if (i >= lo) { zc = -(es[i] * buf[u]) * zc; zk[(size_t)i * M] = zc; }
                }
            }
        }
        // from the twist up
        {
            double zc = 1.0;
            for (int i0 = r; i0 < hi; i0 += BIG_PF) {
                double buf[BIG_PF];
#pragma unroll
                for (int u = 0; u < BIG_PF; ++u) buf[u] = (i0 + u < hi) ? zk[(size_t)(i0 + u + 1) * M] : 0.0;
#pragma unroll
                for (int u = 0; u < BIG_PF; ++u) {
                    const int i = i0 + u;
                    if (i < hi) { zc = -(es[i] * buf[u]) * zc; zk[(size_t)(i + 1) * M] = zc; }
                }
            }
        }
        double n0 = 0.0, n1 = 0.0;
        for (int i0 = lo; i0 <= hi; i0 += BIG_PF) {
            double buf[BIG_PF];
#pragma unroll
            for (int u = 0; u < BIG_PF; ++u) buf[u] = (i0 + u <= hi) ? zk[(size_t)(i0 + u) * M] : 0.0;
#pragma unroll
            for (int u = 0; u < BIG_PF; u += 2) { n0 = fma(buf[u], buf[u], n0); n1 = fma(buf[u + 1], buf[u + 1], n1); }
        }
        const double sc = rsqrt(n0 + n1);
        double r2 = 0.0, zm = 0.0, zmm = 0.0;            // z[i-1], z[i-2]
        for (int i0 = lo; i0 <= hi; i0 += BIG_PF) {
            double buf[BIG_PF];
#pragma unroll
            for (int u = 0; u < BIG_PF; ++u) buf[u] = (i0 + u <= hi) ? zk[(size_t)(i0 + u) * M] : 0.0;
#pragma unroll
            for (int u = 0; u < BIG_PF; ++u) {
                const int i = i0 + u;
                if (i <= hi) {
                    const double zi = buf[u] * sc;
                    zk[(size_t)i * M] = zi;
                    if (i > lo) {                         // residual row i - 1 is complete once z[i] is known
                        const double up = (i > lo + 1) ? es[i - 2] * zmm : 0.0;
                        const double t = fma(ds[i - 1] - lam, zm, fma(es[i - 1], zi, up));
                        r2 = fma(t, t, r2);
                    }
                    zmm = zm; zm = zi;
                }
            }
        }
        {
            const double t = fma(ds[hi] - lam, zm, es[hi - 1] * zmm);
            r2 = fma(t, t, r2);
        }
        res = sqrt(r2);
        for (int i = 0; i < lo; ++i) zk[(size_t)i * M] = 0.0;
        for (int i = hi + 1; i < M; ++i) zk[(size_t)i * M] = 0.0;
    } else if (k < M) {
        for (int i = 0; i < M; ++i) Z[(size_t)i * M + k] = (i == k) ? 1.0 : 0.0;
    }
    // anything suspicious hands the matrix to the classic iteration (generic_apply)
    const bool bad = !(res <= 64.0 * eps * nrm * sqrt((double)M));
    if (__syncthreads_or(bad ? 1 : 0)) {
        if (k == 0) ws.flags[b] = FLAG_SLOW;
        return;
    }
    // eigenvalues closer than GV_GAP ||T|| inside a block: first-order symmetric orthogonalisation,
    // z_k -= 1/2 (z_q . z_k) z_q for every such partner q, all from the uncorrected vectors: the
    // coefficients first (reads only), then row by row -- read, barrier, write
    const double gapabs = GV_GAP * nrm;
    PartnerList pl;
    if (own) {
        const int s0 = inv[k];
        for (int t = 1; s0 - t >= 0 && lam - wsrt[s0 - t] < gapabs; ++t) {
            const int q = perm[s0 - t];
            if (q >= lo && q <= hi) pl.add(q);
        }
        for (int t = 1; s0 + t < M && wsrt[s0 + t] - lam < gapabs; ++t) {
            const int q = perm[s0 + t];
            if (q >= lo && q <= hi) pl.add(q);
        }
    }
    if (!__syncthreads_or(pl.np)) return;
    // Eight rows of Z at a time pass through shared memory (one coalesced copy per tile; the partners'
    // entries are then random reads of the tile, not of L2): first the coefficients -1/2 z_q . z_k, kept in
    // shared memory, then z_k += sum_q h_q z_q tile by tile -- the tile holds the uncorrected rows, so the
    // corrected ones go straight back to Z.
    const int np = pl.np, NTc = blockDim.x;
    constexpr int TR = 8;
    double* tile = reinterpret_cast<double*>(inv + M);                  // [TR][M] (perm and inv: 2 M ints)
    double* hc = tile + (size_t)TR * M;                                  // [2 GV_PH][NTc]
    for (int t = 0; t < np; ++t) hc[t * NTc + k] = 0.0;
    for (int i0 = 0; i0 < M; i0 += TR) {
        __syncthreads();
        for (int idx = k; idx < TR * M; idx += NTc) {
            const int u = idx / M, c = idx - u * M;
            tile[idx] = (i0 + u < M) ? Z[(size_t)(i0 + u) * M + c] : 0.0;
        }
        __syncthreads();
        for (int t = 0; t < np; ++t) {
            const int q = pl.get(t);
            double d0 = 0.0, d1 = 0.0;
#pragma unroll
            for (int u = 0; u < TR; u += 2) {
                d0 = fma(tile[u * M + k], tile[u * M + q], d0);
                d1 = fma(tile[(u + 1) * M + k], tile[(u + 1) * M + q], d1);
            }
            hc[t * NTc + k] += d0 + d1;
        }
    }
    for (int i0 = 0; i0 < M; i0 += TR) {
        __syncthreads();
        for (int idx = k; idx < TR * M; idx += NTc) {
            const int u = idx / M, c = idx - u * M;
            tile[idx] = (i0 + u < M) ? Z[(size_t)(i0 + u) * M + c] : 0.0;
        }
        __syncthreads();
        if (np > 0) {
            double nz[TR];
#pragma unroll
            for (int u = 0; u < TR; ++u) nz[u] = tile[u * M + k];
            for (int t = 0; t < np; ++t) {
                const int q = pl.get(t);
                const double h = -0.5 * hc[t * NTc + k];
#pragma unroll
                for (int u = 0; u < TR; ++u) nz[u] = fma(h, tile[u * M + q], nz[u]);
            }
#pragma unroll
            for (int u = 0; u < TR; ++u)
                if (i0 + u < M) Z[(size_t)(i0 + u) * M + k] = nz[u];
        }
    }
}

// V^T = Z^T B with B = Q^T as the reduction kernels left it in the output buffer (Qt layout), one CTA
// of 8 warps per matrix.  Output columns (= rows of V) are taken CB = 8 CT at a time: the block
// B[:, c0 .. c0 + CB) sits in shared memory (stride CB + 4), Z streams through in chunks of 16 rows
// (cp.async, double-buffered, stride MP + 4: both operands are read as "lane l: [4 kk + l % 4][8 tile +
// l / 4]", conflict-free with a stride of 4 mod 16 doubles), warp w accumulates the 8-row tiles w,
// w + 8, ... of V^T (RTW of them) over all CT column tiles.  The block then passes through shared
// memory once more, transposed and with its columns in ascending order of the eigenvalues, and
// leaves as whole rows of V: straight into the output buffer when one block covers the matrix
// (M <= 128: B is entirely on chip by then), else into the staging area, which is copied over the
// output buffer at the end.
template <int RTW, int CT>
__global__ void __launch_bounds__(BIG_NT)
big_gemm(double* __restrict__ V_, Workspace ws, int M)
{
    constexpr int CB = 8 * CT, LDB = CB + 4, KC = 16;
    extern __shared__ __align__(16) double bg_sm[];
    const int MP = (M + 15) & ~15, LDZ = MP + 4, RT = MP / 8;
    double* Bs = bg_sm;                                   // [MP][LDB], later the output block [CB][LDO]
    double* Zs = Bs + (size_t)MP * LDB;                   // [2][KC][LDZ]
    int* inv = reinterpret_cast<int*>(Zs + 2 * KC * LDZ); // [M]
    const size_t b = blockIdx.x;
    if (ws.flags[b] != FLAG_GETVEC) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double* Z = big_z(ws, b);
    double* V = V_ + b * (size_t)M * M;
    const int nblk = (M + CB - 1) / CB;
    double* Out = (nblk == 1) ? V : big_z(ws, b) + (size_t)M * M;
    const int LDO = M | 1;
    for (int k = tid; k < M; k += BIG_NT) inv[ws.perm[b * M + k]] = k;

    auto stage_z = [&](int chunk, int buf) {              // rows 16 chunk ... of Z, zero beyond M
        double* dst = Zs + (size_t)buf * KC * LDZ;
        const int i0 = chunk * KC;
        for (int idx = tid; idx < KC * MP; idx += BIG_NT) {
            const int ii = idx / MP, kk = idx - ii * MP;
            if (i0 + ii < M && kk < M) cp_async8(dst + ii * LDZ + kk, Z + (size_t)(i0 + ii) * M + kk);
            else dst[ii * LDZ + kk] = 0.0;
        }
    };
    const int nchunk = MP / KC;
    for (int blk = 0; blk < nblk; ++blk) {
        const int c0 = blk * CB;
        __syncthreads();                                  // the output block of the previous round has left
        stage_z(0, 0);
        for (int idx = tid; idx < MP * CB; idx += BIG_NT) {
            const int i = idx / CB, c = idx - i * CB;
            Bs[i * LDB + c] = (i < M && c0 + c < M) ? V[(size_t)i * M + c0 + c] : 0.0;
        }
        double acc[RTW][CT][2];
#pragma unroll
        for (int t = 0; t < RTW; ++t)
#pragma unroll
            for (int ct = 0; ct < CT; ++ct) { acc[t][ct][0] = 0.0; acc[t][ct][1] = 0.0; }
        cp_async_wait_all();
        __syncthreads();
        for (int ch = 0; ch < nchunk; ++ch) {
            if (ch + 1 < nchunk) stage_z(ch + 1, (ch + 1) & 1);
            const double* zs = Zs + (size_t)(ch & 1) * KC * LDZ + (lane & 3) * LDZ + (lane >> 2);
            const double* bs = Bs + (size_t)(ch * KC + (lane & 3)) * LDB + (lane >> 2);
#pragma unroll
            for (int kk = 0; kk < KC / 4; ++kk) {
                double a[RTW];
#pragma unroll
                for (int t = 0; t < RTW; ++t) {
                    const int rt = warp + 8 * t;
                    a[t] = (rt < RT) ? zs[4 * kk * LDZ + 8 * rt] : 0.0;
                }
#pragma unroll
                for (int ct = 0; ct < CT; ++ct) {
                    const double bv = bs[4 * kk * LDB + 8 * ct];
#pragma unroll
                    for (int t = 0; t < RTW; ++t) dmma884(acc[t][ct], a[t], bv);
                }
            }
            cp_async_wait_all();
            __syncthreads();
        }
        // acc[t][ct] = V^T[8 rt + l/4][c0 + 8 ct + 2 (l%4) + {0, 1}] -> Out block [c][inv[k]]
        double* Ob = Bs;
#pragma unroll
        for (int t = 0; t < RTW; ++t) {
            const int kq = 8 * (warp + 8 * t) + (lane >> 2);
            if (kq < M) {
                const int oc = inv[kq];
#pragma unroll
                for (int ct = 0; ct < CT; ++ct) {
                    const int c = 8 * ct + 2 * (lane & 3);
                    Ob[c * LDO + oc] = acc[t][ct][0];
                    Ob[(c + 1) * LDO + oc] = acc[t][ct][1];
                }
            }
        }
        __syncthreads();
        const int ncols = min(CB, M - c0);
        for (int idx = tid; idx < ncols * M; idx += BIG_NT) {
            const int c = idx / M, x = idx - c * M;
            Out[(size_t)(c0 + c) * M + x] = Ob[c * LDO + x];
        }
    }
    if (nblk > 1) {
        __syncthreads();
        const double* src = Out;
        for (int idx = tid; idx < M * M; idx += BIG_NT) V[idx] = src[idx];
    }
}

template <int CT> static inline size_t big_gemm_smem(int M)
{
    const int MP = (M + 15) & ~15;
    return sizeof(double) * ((size_t)MP * (8 * CT + 4) + 2 * 16 * (size_t)(MP + 4)) + sizeof(int) * (size_t)M + 16;
}

}  // namespace letkf

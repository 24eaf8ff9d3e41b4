// ql_kernel.cuh -- step a4: the tridiagonal eigensolver, one THREAD per
// matrix.  PAPER.md:183 (implicit QL as in EISPACK/LAPACK); PAPER.md:204 names the divergence of
// this data-dependent iteration as the efficiency limiter of the paper's warp-per-matrix kernel.
// Here the iteration is taken off the threads that hold the matrix: this kernel runs only the
// O(M^2) scalar recurrences and records the rotations; ql_apply kernels replay them on rows of Q.
#pragma once
#include "common.cuh"

namespace letkf {

constexpr int QL_TPB = 32;   // one warp per CTA: shared memory is 2*M*32 doubles

__global__ void __launch_bounds__(QL_TPB)
ql_log_kernel(Workspace ws, int M, int batch, double* __restrict__ w, int* __restrict__ info)
{
    extern __shared__ double sm[];
    double* dsm = sm;                         // [M][32]
    double* esm = sm + (size_t)M * QL_TPB;    // [M][32]
    const int lane = threadIdx.x;
    const int b0 = blockIdx.x * QL_TPB;
    const int nb = min(QL_TPB, batch - b0);

    // coalesced load of 32 consecutive (d, e) records, transposed into [i][lane]
    for (int idx = lane; idx < QL_TPB * M; idx += QL_TPB) {
        const int bb = idx / M, ii = idx - bb * M;
        double dv = 0.0, ev = 0.0;
        if (bb < nb) {
            dv = ws.dws[(size_t)b0 * M + idx];
            ev = ws.ews[(size_t)b0 * M + idx];
        }
        dsm[ii * QL_TPB + bb] = dv;
        esm[ii * QL_TPB + bb] = ev;
    }
    __syncwarp();

    const int b = b0 + lane;
    double* d = dsm + lane;
    double* e = esm + lane;
    int overflow = 0;
    int nsw = 0;
    int nrot = 0;
    QLState st{0, 0, 0};
    if (lane < nb) {
        e[(size_t)(M - 1) * QL_TPB] = 0.0;
        double2* rot = ws.rot + (size_t)b * ws.logcap;
        uint32_t* hdr = ws.hdr + (size_t)b * ws.swcap;
        int pos = 0;
        for (;;) {
            int lo, m;
            const int rc = ql_next_sweep(st, d, e, QL_TPB, M, rot + pos, ws.logcap - pos, lo, m);
            if (rc == 0) break;
            if (rc < 0 || nsw >= ws.swcap) { overflow = 1; break; }
            hdr[nsw++] = (uint32_t)lo | ((uint32_t)m << 16);
            pos += m - lo;
        }
        if (!overflow) sort_eigenvalues(d, QL_TPB, reinterpret_cast<int*>(e), QL_TPB * 2, M);
        ws.nsweeps[b] = nsw;
        ws.flags[b] = overflow;
        if (info && !overflow) info[b] = st.fail;
        nrot = pos;
    }
    __syncwarp();
    if (ws.rot_counter) {
        const int tot = __reduce_add_sync(0xffffffffu, nrot);
        if (lane == 0) atomicAdd(ws.rot_counter, (unsigned long long)tot);
    }
    // coalesced store of w and perm (matrices that overflowed are rewritten by the slow path)
    const int* psm = reinterpret_cast<const int*>(esm);
    for (int idx = lane; idx < QL_TPB * M; idx += QL_TPB) {
        const int bb = idx / M, ii = idx - bb * M;
        if (bb < nb) {
            w[(size_t)b0 * M + idx] = dsm[ii * QL_TPB + bb];
            ws.perm[(size_t)b0 * M + idx] = psm[(ii * QL_TPB + bb) * 2];
        }
    }
}

}  // namespace letkf

// ql_kernel.cuh -- step a4: the tridiagonal eigensolver, one THREAD per
// matrix.  PAPER.md:183 (implicit QL as in EISPACK/LAPACK); PAPER.md:204 names the divergence of
// this data-dependent iteration as the efficiency limiter of the paper's warp-per-matrix kernel.
// Here the iteration is taken off the threads that hold the matrix: this kernel runs only the
// O(M^2) scalar recurrences and records the rotations; the apply kernels replay them on rows of Q.
//
// The 32 matrices of a warp advance in LOCKSTEP: every pass, each lane sets up its next sweep
// (deflation scan + Wilkinson shift), then the warp runs max-over-lanes rotation steps with the
// shorter sweeps predicated off.  All loop bounds are warp-uniform (votes), so the lanes never
// fall into the serialised divergence that a per-lane while-loop produces (measured: 1.4 active
// threads per instruction before this restructuring, profiles/).
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
    const unsigned FULL = 0xffffffffu;
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
    const bool valid = lane < nb;
    double* d = dsm + lane;
    double* e = esm + lane;
    constexpr int stride = QL_TPB;
    e[(size_t)(M - 1) * stride] = 0.0;
    double2* rot = ws.rot + (size_t)(valid ? b : b0) * ws.logcap;
    uint32_t* hdr = ws.hdr + (size_t)(valid ? b : b0) * ws.swcap;

    QLState st{0, 0, 0};
    int overflow = 0, nsw = 0, pos = 0;
    bool done = !valid;
    for (;;) {
        // ---- per-lane sweep set-up (divergent inside, reconverges at the vote)
        int l = 0, m = 0, i = -1;
        double g = 0.0, s = 1.0, c = 1.0, p = 0.0;
        bool sweeping = false;
        if (!done) {
            if (ql_find_block(st, d, e, stride, M, m)) {
                l = st.l;
                if (pos + (m - l) > ws.logcap || nsw >= ws.swcap) { overflow = 1; done = true; }
                else { g = ql_shift(d, e, stride, l, m); i = m - 1; sweeping = true; }
            } else {
                done = true;
            }
        }
        if (!__any_sync(FULL, sweeping)) break;
        const int maxlen = __reduce_max_sync(FULL, sweeping ? m - l : 0);
        // ---- lockstep rotation steps
        bool broke = false;
        for (int k = 0; k < maxlen; ++k) {
            if (sweeping && !broke && i >= l) {
                double2 cs;
                if (ql_rot_step(d, e, stride, i, m, s, c, p, g, cs)) {
                    rot[pos + (m - 1 - i)] = cs;
                    --i;
                } else {
                    broke = true;
                }
            }
        }
        if (sweeping) {
            int lo;
            if (broke) lo = i + 1;
            else { ql_finish_sweep(d, e, stride, l, m, p, g); lo = l; }
            if (m - lo > 0) {
                hdr[nsw++] = (uint32_t)lo | ((uint32_t)m << 16);
                pos += m - lo;
            }
        }
    }
    if (valid) {
        if (!overflow) sort_eigenvalues(d, QL_TPB, reinterpret_cast<int*>(e), QL_TPB * 2, M);
        ws.nsweeps[b] = nsw;
        ws.flags[b] = overflow;
        if (info && !overflow) info[b] = st.fail;
    }
    __syncwarp();
    if (ws.rot_counter) {
        const int tot = __reduce_add_sync(FULL, valid ? pos : 0);
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

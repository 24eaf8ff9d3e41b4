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

// QL_TPB matrices per CTA (a multiple of 32; each warp is its own lockstep group): shared memory is
// 2*M*QL_TPB doubles.  Several warps per CTA do not make the kernel faster -- they make the CTAs
// fewer and larger, so that a QL CTA arriving on an SM full of tridiag / apply CTAs evicts ONE of
// them for up to three warps of QL work instead of one per warp (Streams).
//
// two_pass (large batches, where the replay is what costs): the iteration is run TWICE, by the two
// lanes of a pair.  The even lane (Wilkinson shifts, nothing logged) only finds the eigenvalues; the
// odd lane works on a copy of its own and shifts the first sweep for position l by the eigenvalue
// its partner has found there (a "perfect" shift: in exact arithmetic one sweep deflates it),
// falling back to Wilkinson shifts for any further sweep; it waits at position l until the partner
// has passed it.  The logged sequence is 31-40% shorter (measured on the configured workloads: 1.83
// -> 1.32 sweeps per eigenvalue, 1.05 M^2 -> 0.73 M^2 rotations at M = 64) and every rotation saved
// is 6 M flops saved in the replay, while the latency stays that of ONE pass (the two run side by
// side, the second a few sweeps behind).  The result is an orthogonal similarity either way.
//
// modes 2 and 3 (M <= 64, the register path): ONE lane per matrix.  QL_CLASSIFY runs the eigenvalue-
// only pass and then CLASSIFIES the matrix (common.cuh, GV_*): if its eigenvalues are separated well
// enough for the apply kernel to form the eigenvectors of T directly (twisted factorisations),
// nothing is ever logged (flags[b] = FLAG_GETVEC); otherwise the eigenvalues are left by position in
// ws.s1 and the matrix is marked FLAG_PENDING.  QL_LOGPASS (a second launch, the first one that needs
// the matrix's slot of the rotation log) runs the logging pass of the pending matrices, shifted by
// those eigenvalues (-> FLAG_REPLAY); a CTA without a pending matrix leaves at once.
constexpr int QL_ONE_PASS = 0, QL_TWO_PASS = 1, QL_CLASSIFY = 2, QL_LOGPASS = 3, QL_LOGPASS_PAIRED = 4, QL_PAIRED_CLASSIFY = 5;
// (QL_LOGPASS_PAIRED: the pending matrices as in QL_LOGPASS, but by pairs of lanes as in QL_TWO_PASS --
// behind bisect_kernel.cuh, whose eigenvalues are not in the order in which QL would deflate them;
// QL_PAIRED_CLASSIFY (M > 64, big_kernels.cuh): QL_TWO_PASS, and the matrix is classified at the end -- easy: FLAG_GETVEC, the
// log is dropped (its record becomes the store of the eigenvectors of T); else FLAG_REPLAY.  One launch and the latency of one
// pass whatever the spectrum, at the price of log writes nobody reads for the easy matrices)

// The mode is a template parameter: in the eigenvalue-only pass the log stores, the shift look-up and the
// pair bookkeeping are not compiled in at all (as run-time predicates they cost 30% of the rotation step).
template <int QL_TPB, int mode>
__global__ void __launch_bounds__(QL_TPB, 1024 / QL_TPB)     // <= 64 registers: a QL CTA arriving beside tridiag / apply CTAs must stay small
ql_log_kernel(Workspace ws, int M, int batch, double* __restrict__ w, int* __restrict__ info)
{
    extern __shared__ double sm[];
    double* dsm = sm;                             // [M][QL_TPB]  one column per LANE
    double* esm = sm + (size_t)M * QL_TPB;        // [M][QL_TPB]
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x;              // column of the [M][QL_TPB] arrays
    constexpr bool two_pass = mode == QL_TWO_PASS || mode == QL_LOGPASS_PAIRED || mode == QL_PAIRED_CLASSIFY;  // (pairs of lanes)
    constexpr bool classify = mode == QL_CLASSIFY || mode == QL_PAIRED_CLASSIFY;
    constexpr bool pending_only = mode == QL_LOGPASS || mode == QL_LOGPASS_PAIRED;
    const int nmc = two_pass ? QL_TPB / 2 : QL_TPB;         // matrices per CTA
    const int b0 = blockIdx.x * nmc;
    const int nb = min(nmc, batch - b0);

    // coalesced load of the CTA's (d, e) records, transposed into [i][lane] (two_pass: both lanes of a pair)
    for (int idx = lane; idx < nmc * M; idx += QL_TPB) {
        const int bb = idx / M, ii = idx - bb * M;
        double dv = 0.0, ev = 0.0;
        if (bb < nb) {
            dv = ws.dws[(size_t)b0 * M + idx];
            ev = ws.ews[(size_t)b0 * M + idx];
        }
        if (two_pass) {
            dsm[ii * QL_TPB + 2 * bb] = dv;     esm[ii * QL_TPB + 2 * bb] = ev;
            dsm[ii * QL_TPB + 2 * bb + 1] = dv; esm[ii * QL_TPB + 2 * bb + 1] = ev;
        } else {
            dsm[ii * QL_TPB + bb] = dv;
            esm[ii * QL_TPB + bb] = ev;
        }
    }
    __syncthreads();

    const int mloc = two_pass ? lane >> 1 : lane;            // matrix of this lane within the CTA
    const int b = b0 + mloc;
    bool valid = mloc < nb;
    if (pending_only) {                                      // only the matrices the classifier left pending
        valid = valid && ws.flags[b] == FLAG_PENDING;
        if (!__syncthreads_or(valid ? 1 : 0)) return;
    }
    const bool logging = mode == QL_ONE_PASS || mode == QL_LOGPASS || (two_pass && (lane & 1));   // rotations recorded
    bool easy = false;                                       // QL_CLASSIFY: FLAG_GETVEC
    constexpr bool shifted = two_pass || mode == QL_LOGPASS;     // first sweep of a position shifted by a known eigenvalue
    double* d = dsm + lane;
    double* e = esm + lane;
    constexpr int stride = QL_TPB;
    e[(size_t)(M - 1) * stride] = 0.0;
    double2* rot = ws.rot + (size_t)(valid ? b : b0) * ws.logcap;
    uint32_t* hdr = ws.hdr + (size_t)(valid ? b : b0) * ws.swcap;
    // eigenvalues of the first pass, by position: the partner's diagonal (pairs of lanes), or ws.s1
    double* s1g = ws.s1 + (size_t)(valid ? b : b0) * M;
    const int swcap = ws.swcap;

    // Per-lane state: the unreduced block [l, m] (e[m] == 0), the sweeps spent on eigenvalue l,
    // the failures.  The deflation test of the classic algorithm ("first m >= l with negligible
    // e[m]", rescanned before every sweep) is evaluated INSIDE the sweep on the values it has
    // just produced, so the per-sweep rescan disappears (it was 30% of this kernel, profiles/r01a);
    // a scan is needed only when l enters a part of the matrix no sweep of this block has seen.
    const double eps = 1.1102230246251565e-16;   // 2^-53 (reading G10)
    const double thr = valid ? ql_threshold(d, e, stride, M) : 0.0;   // 2^-53 max_i(|d_i| + |e_i|)
#define QL_D(i) d[(i) * stride]
#define QL_E(i) e[(i) * stride]
    auto scan_end = [&](int from) {
        int k = from;
        for (; k < M - 1; ++k)
            if (fabs(QL_E(k)) <= fmax(eps * (fabs(QL_D(k)) + fabs(QL_D(k + 1))), thr)) break;
        QL_E(k) = 0.0;
        return k;
    };
    // the split of the input (reading G24, common.cuh: GV_SPLIT): negligible off-diagonals are exactly 0 from here on;
    // mode 2 keeps the boundaries of the unreduced blocks (bit i: e_i = 0), nw64 words per lane behind the (d, e) arrays
    const int nw64 = (M + 63) >> 6;
    unsigned long long* bm_sh = reinterpret_cast<unsigned long long*>(sm + 2 * (size_t)M * QL_TPB);   // [nw64][QL_TPB]
    if (valid) {
        unsigned long long word = 0ull;
        for (int k = 0; k < M - 1; ++k) {
            if (fabs(QL_E(k)) <= fmax(eps * (fabs(QL_D(k)) + fabs(QL_D(k + 1))), GV_SPLIT * thr)) { QL_E(k) = 0.0; word |= 1ull << (k & 63); }
            if (classify && ((k & 63) == 63 || k == M - 2)) { bm_sh[(k >> 6) * QL_TPB + lane] = word; word = 0ull; }
        }
        if (classify && M == 1) bm_sh[lane] = 0ull;
    }
    int l = 0, m = 0, iter = 0, fail = 0;
    int overflow = 0, nsw = 0, pos = 0;
    bool done = !valid;
    if (!done) m = scan_end(0);
    for (;;) {
        // progress of the partner lane as of the end of the last round (two_pass)
        __syncwarp();
        const int l_partner = __shfl_xor_sync(FULL, l, 1);
        const bool partner_done = __shfl_xor_sync(FULL, (int)done, 1) != 0;
        // ---- per-lane sweep set-up (divergent inside, reconverges at the vote)
        bool sweeping = false, waiting = false;
        while (!done) {
            if (m == l) {                              // eigenvalue l has converged
                l += 1; iter = 0;
                if (l >= M) { done = true; break; }
                m = scan_end(l);
                continue;
            }
            if (iter >= QL_MAX_SWEEPS) {               // give up on this one (info counts it)
                fail += 1; QL_E(l) = 0.0; m = l;
                continue;
            }
            if (two_pass && logging && iter == 0 && !(partner_done || l_partner > l)) { waiting = true; break; }
            if (logging && (pos + (m - l) > ws.logcap || nsw >= swcap)) { overflow = 1; done = true; break; }
            iter += 1;
            sweeping = true;
            break;
        }
        if (!__any_sync(FULL, sweeping || waiting)) break;
        int i = -1, mlow = m;
        double g = 0.0, s = 1.0, c = 1.0, p = 0.0, dprev = 0.0;
        if (sweeping) {
            if (shifted && logging && iter == 1) {
                // the eigenvalue the first pass found at position l
                g = QL_D(m) - (two_pass ? dsm[l * stride + (lane ^ 1)] : s1g[l]);
            } else {
                // Wilkinson shift
                const double el = QL_E(l), dl = QL_D(l);
                const double gg = (QL_D(l + 1) - dl) / (2.0 * el);
                const double rr = sqrt(gg * gg + 1.0);
                g = QL_D(m) - dl + el / (gg + copysign(rr, gg));
            }
            i = m - 1;
        }
        const int maxlen = __reduce_max_sync(FULL, sweeping ? m - l : 0);
        // ---- lockstep rotation steps.  The kernel is bound by the dependent chain of one step,
        // g -> r2 = f^2 + g^2 -> 1/sqrt -> c -> g, and the SM issues in order, so whatever else a
        // step computes must not stand between two links of that chain, and the step must be ONE
        // basic block for ptxas to interleave the rest with it.  Hence:
        //  * the step is software-pipelined by hand: p, the new d, its store and the deflation test
        //    of step i+1 are computed at the top of step i, in the shadow of the 1/sqrt of step i;
        //  * r is formed as q/r with q = g tb + (d_i - gt) f, known before 1/r is;
        //  * the operands of step i-1 are loaded at the top of step i;
        //  * 1/sqrt is the hardware seed (2^-20) and one third-order step (measured 49 cycles
        //    against 63 for two Newton steps, same 2.7e-16 error);
        //  * no branch for the rare cases: an r2 outside [1e-280, 1e280] (underflow to the block
        //    split of the classic algorithm, overflow, NaN) only sets a flag; the sweep runs on
        //    garbage in the lane's own shared memory, and the matrix is handed to the slow path
        //    (flags[b], like a log overflow), whose step treats those cases one by one.
        double2* outp = rot + pos;
        double* pd = d + (i > 0 ? i : 0) * stride;     // &d[i]
        double* pe = e + (i > 0 ? i : 0) * stride;     // &e[i]
        double ei = 0.0, di = 0.0, di1 = 0.0;
        double rp = 0.0, gtp = 0.0, enp = 0.0;         // r, gt and new e of the step before (pending)
        bool bad = false;
        if (sweeping) { ei = pe[0]; di = pd[0]; di1 = pd[stride]; gtp = pd[2 * stride]; }
        auto step = [&]() {
            {
                const int nxt = (i > l) ? -stride : 0;
                const double ein = pe[nxt], din = pd[nxt];
                const double f = s * ei;
                const double b2 = c * ei;
                const double tb = b2 + b2;
                const double r2 = fma(f, f, g * g);
                double rinv;
                asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(rinv) : "d"(r2));
                // exponent of r2 in [2^-930, 2^930), on the integer pipe
                bad |= ((unsigned)__double2hiint(r2) - 0x05d00000u) >= 0x74400000u;
                // in the shadow: finish step i+1 (s is still its s) ...
                // (at the first step of a sweep nothing is pending: rp = 0, gtp = the value at d[m+1]
                // -- or, for m = M-1, at the word that follows the d array -- which is written back)
                p = s * rp;
                const double dnew = gtp + p;
                if (sweeping) pd[2 * stride] = dnew;
                // ... its deflation test, on this sweep's values (d[i+3] = dprev):
                // |e| <= max(eps (|d| + |d'|), thr)  <=>  2^53 |e| <= |d| + |d'|  or  |e| <= thr
                const double es = __hiloint2double(__double2hiint(enp) + (53 << 20), __double2loint(enp));
                const bool defl = (i + 2 < m) & ((fabs(es) <= fabs(dnew) + fabs(dprev)) | (fabs(enp) <= thr));   // no short circuit: no branch
                mlow = defl ? i + 2 : mlow;
                dprev = dnew;
                // ... and what this step can form without 1/r
                const double gt = di1 - p;
                const double q = fma(g, tb, (di - gt) * f);
                {
                    // (one = 1 + 0 q ties q to the MIDDLE of the 1/sqrt chain: ptxas otherwise sinks
                    // the five operations of q behind 1/r, where they add 16 cycles to the chain;
                    // 0 q is not folded because q may be NaN -- when it is, so is the result)
                    const double one = fma(q, 0.0, 1.0);
                    const double t = fma(-(0.5 * r2) * rinv, rinv, 0.5);
                    const double u = fma(1.5, t, one);
                    rinv = fma(rinv * t, u, rinv);
                }
                s = f * rinv;
                c = g * rinv;
                rp = q * rinv;
                g = fma(c, rp, -b2);
                enp = r2 * rinv;
                gtp = gt;
                if (sweeping) pe[stride] = enp;
                if (sweeping && logging) *outp = make_double2(c, s);
                ++outp;
                di1 = di; di = din; ei = ein;
                pd += nxt; pe += nxt;
                --i;
            }
        };
        // the first minlen steps are taken by every sweeping lane: no per-lane guard, hence no
        // divergence construct around the step (BSSY / BRA / BSYNC and the latency of the
        // reconvergence cost ~40 of a step's ~200 cycles); lanes that are not sweeping ride along on
        // their own column with their stores predicated off.  Only the ragged rest is guarded.
        const int minlen = __reduce_min_sync(FULL, sweeping ? m - l : 0x7fffffff);
        int k = 0;
        for (; k < minlen && k < maxlen; ++k) step();
        for (; k < maxlen; ++k)
            if (i >= l) step();                        // (i = l - 1 when the lane's sweep is done)
        if (sweeping) {
            if (bad) {                                 // left to the slow path
                overflow = 1; done = true;
            } else {
                // the last step (i = l) is still pending
                p = s * rp;
                const double dnew = gtp + p;
                QL_D(l + 1) = dnew;
                if (l + 1 < m && fabs(enp) <= fmax(eps * (fabs(dnew) + fabs(dprev)), thr)) mlow = l + 1;
                dprev = dnew;
                const double dl = QL_D(l) - p;
                QL_D(l) = dl;
                QL_E(l) = g;
                QL_E(m) = 0.0;
                if (logging) {
                    hdr[nsw++] = (uint32_t)l | ((uint32_t)m << 16);
                    pos += m - l;
                }
                if (mlow < m) QL_E(mlow) = 0.0;
                m = mlow;
                // eigenvalue l converged: the next block starts at l+1 and ends at mlow, the lowest
                // negligible off-diagonal this sweep has seen above l -- no rescan
                if (fabs(g) <= fmax(eps * (fabs(dl) + fabs(dprev)), thr)) { QL_E(l) = 0.0; l += 1; iter = 0; }
            }
        }
    }
#undef QL_D
#undef QL_E
    // ---- the eigenvalues of every matrix of the CTA are sorted by ALL its lanes together (rank of
    // lambda_k = number of eigenvalues below it: no dependent chain; one lane sorting its own matrix
    // by insertion was 28% of this kernel), and in QL_CLASSIFY the sorted sequence is classified on
    // the way (common.cuh, GV_*): easy unless two eigenvalues that are not both 1 x 1 blocks are
    // closer than GV_TINY ||T||, or more than GV_PH lie within GV_GAP ||T|| above one.
    // The lanes work in groups of GS = 16 / 32 / 64 >= M (M <= 64), one matrix per group and round:
    // QL_TPB / GS matrices per round (at M = 16 one matrix per round left 112 of 128 lanes idle through
    // 128 rounds of three barriers each -- more than the iteration itself took).
    const bool owner = valid && (!two_pass || (lane & 1));   // the lane that reports the matrix
    double* thr_sh = reinterpret_cast<double*>(bm_sh + (size_t)nw64 * QL_TPB);                         // [QL_TPB]
    int* sort_sh = reinterpret_cast<int*>(thr_sh + QL_TPB);                                            // [QL_TPB] 1: to sort, 2: and hard
    sort_sh[lane] = (owner && !overflow) ? 1 : 0;
    thr_sh[lane] = thr;
    __syncthreads();
    const int gs0 = M <= 16 ? 16 : (M <= 32 ? 32 : 64);
    const int GS = (M <= 64 && QL_TPB % gs0 == 0) ? gs0 : QL_TPB;      // lanes per matrix
    const int ng = QL_TPB / GS, grp = lane / GS, kl = lane - grp * GS;
    constexpr int KMAX = 8;                                   // eigenvalues per lane: M <= 256 = KMAX * 32
    for (int c0 = 0; c0 < nb; c0 += ng) {
        const int c = c0 + grp;
        const int col = two_pass ? 2 * c + 1 : c;
        const bool act = c < nb && sort_sh[col] != 0;
        const size_t bc = (size_t)(b0 + c);
        const double* dc = dsm + (act ? col : 0);
        double* ec = esm + (act ? col : 0);
        int myrank[KMAX];
#pragma unroll
        for (int t = 0; t < KMAX; ++t) {
            const int k = kl + t * GS;
            myrank[t] = -1;
            if (act && k < M) {
                const double v = dc[k * stride];
                int rank = 0;
                for (int j = 0; j < M; ++j) {
                    const double u = dc[j * stride];
                    rank += (u < v || (u == v && j < k)) ? 1 : 0;
                }
                w[bc * M + rank] = v;
                ws.perm[bc * M + rank] = k;
                if (classify) { ws.s1[bc * M + k] = v; ec[rank * stride] = v; myrank[t] = rank; }
            }
        }
        if (classify) {
            __syncthreads();
#pragma unroll
            for (int t = 0; t < KMAX; ++t) {
                const int k = kl + t * GS;
                if (act && k < M) {
                    // block of position k: first position behind the last boundary below k; id > 0, negated for a 1 x 1 block
                    int lo = 0;
                    if (k > 0) {
                        int wq = (k - 1) >> 6;
                        unsigned long long bits = bm_sh[wq * QL_TPB + col] & (~0ull >> (63 - ((k - 1) & 63)));
                        while (bits == 0ull && wq > 0) { --wq; bits = bm_sh[wq * QL_TPB + col]; }
                        if (bits) lo = 64 * wq + (63 - __clzll((long long)bits)) + 1;
                    }
                    const bool hi_cut = k == M - 1 || ((bm_sh[(k >> 6) * QL_TPB + col] >> (k & 63)) & 1ull);
                    dsm[myrank[t] * stride + col] = (lo == k && hi_cut) ? -(double)(lo + 1) : (double)(lo + 1);
                }
            }
            __syncthreads();
            bool hard = false;
            if (act) {
                const double nrm = thr_sh[col] * 9007199254740992.0;               // max_i(|d_i| + |e_i|)
                for (int k = kl; k + 1 < M && !hard; k += GS)                       // sorted index
                    hard = gv_hard_at(k, M, nrm, [&](int u) { return ec[u * stride]; }, [&](int u) { return (int)dc[u * stride]; });
            }
            if (hard) sort_sh[col] = 2;                       // (every writer writes the same value)
        }
    }
    if (classify) {
        __syncthreads();
        easy = sort_sh[lane] == 1;
    }
    if (owner) {
        ws.nsweeps[b] = nsw;
        ws.flags[b] = overflow ? FLAG_SLOW : (classify && easy ? FLAG_GETVEC : (mode == QL_CLASSIFY ? FLAG_PENDING : FLAG_REPLAY));
        if (info && !overflow) info[b] = fail;
    }
    if (ws.rot_counter) {
        const int tot = __reduce_add_sync(FULL, (valid && logging && !easy) ? pos : 0);   // (a log that is dropped does not count)
        if ((lane & 31) == 0) atomicAdd(ws.rot_counter, (unsigned long long)tot);
        const int ne = __reduce_add_sync(FULL, (owner && easy) ? 1 : 0);
        if ((lane & 31) == 0 && ne) atomicAdd(ws.rot_counter + 1, (unsigned long long)ne);
    }
}

}  // namespace letkf

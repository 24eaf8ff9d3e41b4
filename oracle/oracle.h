/*
 * oracle.h -- CPU ORACLE for the LETKF local analysis hot path (arXiv 2308.03310).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path under paper_2308_03310_b200/csrc/ and is
 * never linked into libletkf.  Plain, slow, fp64 (plus an 80-bit long double referee),
 * written so that it can be checked against the paper by eye.
 *
 * What it computes (PAPER.md line numbers; "Eq.n" = the paper's equation n):
 *   oracle_syev*            the EVD "of Q" that PAPER.md:142 asks for: A = V diag(w) V^T,
 *                           V^T V = I, w ascending.  It is the plain definition reached by
 *                           cyclic-by-row Jacobi (a different algorithm family from the
 *                           Householder + QL of PAPER.md:183, on purpose).
 *   oracle_letkf_analysis*  Eq.9-11, Eq.13-17 with
 *                           R^-1 replaced by the diagonal G o R^-1 of PAPER.md:144, and the
 *                           multiplicative inflation rho of ref.[9] (reading G1;
 *                           rho = 1 is Eq.17 exactly).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): known spectrum, 2x2 closed form,
 * tridiagonal Toeplitz closed form, trace/Frobenius invariants, characteristic
 * polynomial brute force (M<=4), Kalman-filter equivalence Eq.6-8, structural
 * identities of W, closed-form special cases, an EVD-free matrix-function route.
 * No function here is "parity unpinned".
 *
 * Layouts: all arrays row-major, batch outermost.
 *   A[batch][M][M], w[batch][M], V[batch][M][M] with eigenvector k in COLUMN k.
 *   Yb[batch][p][M], d[batch][p], rinv_loc[batch][p], Xb[batch][nstate][M],
 *   Xa[batch][nstate][M], W[batch][M][M], wbar[batch][M].
 */
#ifndef LETKF_ORACLE_H
#define LETKF_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

/* One matrix, fp64 Jacobi.  Reads the lower triangle of A (mirrored to a full
 * symmetric work copy).  Returns the number of sweeps used (>=0), or -1 if 60 sweeps
 * did not converge. */
int oracle_syev(const double* A, int M, double* w, double* V);

/* Same algorithm carried out in long double (x87 80-bit, eps ~ 1e-19); inputs and
 * outputs are rounded to double.  The referee when two fp64 results disagree. */
int oracle_syev_ld(const double* A, int M, double* w, double* V);

/* Batch loop (OpenMP over b, "each local problem can be computed in
 * parallel").  info[b] = 0 ok, 1 = no convergence (info may be NULL).
 * nthreads <= 0: OpenMP default.  Returns the number of threads used. */
int oracle_syev_batched(const double* A, int M, int batch, double* w, double* V,
                        int* info, int nthreads);

/* Full local analysis per grid point.  W and wbar may be NULL.  Returns threads used. */
int oracle_letkf_analysis_batched(const double* Yb, const double* d,
                                  const double* rinv_loc, const double* Xb,
                                  int M, int p, int nstate, int batch, double rho,
                                  double* Xa, double* W, double* wbar,
                                  int* info, int nthreads);

/* Localisation function G(dist) of PAPER.md:144 (dist in grid units): loc_kind 0 = Gaussian
 * exp(-dist^2/(2 L^2)) (BASELINE.json), 1 = Gaspari-Cohn with half-width L (zero from 2L on). */
double oracle_localisation(int loc_kind, double L, double dist);

/* Grid form: the local problems of a periodic Ny x Nx grid with the V observed variables of a
 * (2hw+1)^2 patch as local observations (Procedure 1 lines 1-2, Eq.18-19);
 * Yf[V][Ny][Nx][M], yo[V][Ny][Nx], mask[Ny][Nx] or NULL, Xb/Xa[Ny*Nx][nstate][M], wbar may be
 * NULL.  Pinned against the batched form on an explicitly gathered Y_loc
 * (tests/test_oracle_grid.py).  Returns threads used. */
int oracle_letkf_analysis_grid(const double* Yf, const double* yo, const unsigned char* mask,
                               const double* Xb, int M, int V, int Ny, int Nx, int nstate,
                               int hw, int loc_kind, double L, double sigma_o, double rho,
                               double* Xa, double* wbar, int* info, int nthreads);

#ifdef __cplusplus
}
#endif
#endif

/*
 * oracle.c -- CPU ORACLE (test infrastructure, see oracle.h).  Plain C99, fp64.
 * Nothing here is tuned; nothing here is shared with the CUDA path.
 */
#include "oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- the EVD, twice: fp64 (the oracle) and long double (the referee) ---------------- */
#define REAL double
#define SQRT sqrt
#define FABS fabs
#define JACOBI_NAME jacobi_f64
#include "jacobi_impl.inc"
#undef REAL
#undef SQRT
#undef FABS
#undef JACOBI_NAME

#define REAL long double
#define SQRT sqrtl
#define FABS fabsl
#define JACOBI_NAME jacobi_f80
#include "jacobi_impl.inc"
#undef REAL
#undef SQRT
#undef FABS
#undef JACOBI_NAME

int oracle_syev(const double* A, int M, double* w, double* V)
{
    double* S;
    int sweeps;
    if (M < 1) return 0;
    S = (double*)malloc(sizeof(double) * (size_t)M * M);
    sweeps = jacobi_f64(A, M, S, V, w);
    free(S);
    return sweeps;
}

int oracle_syev_ld(const double* A, int M, double* w, double* V)
{
    long double *S, *VV, *ww;
    int sweeps, i;
    if (M < 1) return 0;
    S  = (long double*)malloc(sizeof(long double) * (size_t)M * M);
    VV = (long double*)malloc(sizeof(long double) * (size_t)M * M);
    ww = (long double*)malloc(sizeof(long double) * (size_t)M);
    sweeps = jacobi_f80(A, M, S, VV, ww);
    for (i = 0; i < M; ++i) w[i] = (double)ww[i];
    for (i = 0; i < M * M; ++i) V[i] = (double)VV[i];
    free(S); free(VV); free(ww);
    return sweeps;
}

static int pick_threads(int nthreads)
{
#ifdef _OPENMP
    return (nthreads > 0) ? nthreads : omp_get_max_threads();
#else
    (void)nthreads;
    return 1;
#endif
}

int oracle_syev_batched(const double* A, int M, int batch, double* w, double* V,
                        int* info, int nthreads)
{
    int nt = pick_threads(nthreads);
    long b;
    if (M < 1 || batch < 1) return nt;
#pragma omp parallel for schedule(dynamic) num_threads(nt)
    for (b = 0; b < batch; ++b) {
        int s = oracle_syev(A + b * M * M, M, w + b * M, V + b * M * M);
        if (info) info[b] = (s < 0) ? 1 : 0;
    }
    return nt;
}

/* ---- the local analysis of one grid point ------------------------------------------- */
/*
 * Follows the paper's order and notation:
 *   Q      = ((M-1)/rho) I + dY^T (G o R^-1) dY            Eq.17 (+ rho, reading G1)
 *   g      = dY^T (G o R^-1) (y^o - ybar^f)                right factor of Eq.14
 *   Q      = V diag(lam) V^T
 *   P~a    = Q^-1 = V diag(1/lam) V^T                      Eq.16
 *   wbar^a = P~a g                                         Eq.14
 *   dW^a   = sqrt(M-1) (P~a)^{1/2}
 *          = sqrt(M-1) V diag(lam^-1/2) V^T                Eq.15, symmetric root (reading G2)
 *   xbar   = (1/M) sum_m x_m,  dX = X - xbar               Eq.9-11
 *   x^a_m  = xbar + dX (wbar^a + dw^a_m)                   Eq.13, for each of the nstate
 *                                                          components of the point
 * Inputs: Yb = dY^f as [p][M] (row j = observation j across the ensemble), dvec = y^o - ybar^f,
 * r = diag(G o R^-1), Xb = [nstate][M].
 */
static int analysis_point(const double* Yb, const double* dvec, const double* r,
                          const double* Xb, int M, int p, int ns, double rho,
                          double* Xa, double* W, double* wbar,
                          double* Q, double* g, double* lam, double* V, double* S,
                          double* Wl, double* wb, double* dX)
{
    int m, n, j, k, s, sweeps;

    for (m = 0; m < M; ++m)
        for (n = 0; n < M; ++n) {
            double acc = 0.0;
            for (j = 0; j < p; ++j)
                acc += r[j] * Yb[(long)j * M + m] * Yb[(long)j * M + n];
            Q[(long)m * M + n] = acc + ((m == n) ? (double)(M - 1) / rho : 0.0);
        }
    for (m = 0; m < M; ++m) {
        double acc = 0.0;
        for (j = 0; j < p; ++j)
            acc += Yb[(long)j * M + m] * r[j] * dvec[j];
        g[m] = acc;
    }

    sweeps = jacobi_f64(Q, M, S, V, lam);

    /* wbar = V diag(1/lam) V^T g */
    for (m = 0; m < M; ++m) {
        double acc = 0.0;
        for (k = 0; k < M; ++k) {
            double vtg = 0.0;
            for (n = 0; n < M; ++n) vtg += V[(long)n * M + k] * g[n];
            acc += V[(long)m * M + k] * (1.0 / lam[k]) * vtg;
        }
        wb[m] = acc;
    }
    /* W = sqrt(M-1) V diag(lam^-1/2) V^T */
    for (m = 0; m < M; ++m)
        for (n = 0; n < M; ++n) {
            double acc = 0.0;
            for (k = 0; k < M; ++k)
                acc += V[(long)m * M + k] * (1.0 / sqrt(lam[k])) * V[(long)n * M + k];
            Wl[(long)m * M + n] = sqrt((double)(M - 1)) * acc;
        }
    /* Xa */
    for (s = 0; s < ns; ++s) {
        double xbar = 0.0;
        for (m = 0; m < M; ++m) xbar += Xb[(long)s * M + m];
        xbar /= (double)M;
        for (m = 0; m < M; ++m) dX[m] = Xb[(long)s * M + m] - xbar;
        for (m = 0; m < M; ++m) {
            double acc = 0.0;
            for (k = 0; k < M; ++k)
                acc += dX[k] * (wb[k] + Wl[(long)k * M + m]);
            Xa[(long)s * M + m] = xbar + acc;
        }
    }
    if (W)    memcpy(W, Wl, sizeof(double) * (size_t)M * M);
    if (wbar) memcpy(wbar, wb, sizeof(double) * (size_t)M);
    return sweeps;
}

int oracle_letkf_analysis_batched(const double* Yb, const double* d,
                                  const double* rinv_loc, const double* Xb,
                                  int M, int p, int nstate, int batch, double rho,
                                  double* Xa, double* W, double* wbar,
                                  int* info, int nthreads)
{
    int nt = pick_threads(nthreads);
    if (M < 1 || batch < 1 || nstate < 1 || p < 0) return nt;
#pragma omp parallel num_threads(nt)
    {
        size_t MM = (size_t)M * M;
        double* buf = (double*)malloc(sizeof(double) * (4 * MM + 4 * (size_t)M));
        double *Q = buf, *V = buf + MM, *S = buf + 2 * MM, *Wl = buf + 3 * MM;
        double *g = buf + 4 * MM, *lam = g + M, *wb = lam + M, *dX = wb + M;
        long b;
#pragma omp for schedule(dynamic)
        for (b = 0; b < batch; ++b) {
            int s = analysis_point(Yb + b * (long)p * M, d + b * (long)p,
                                   rinv_loc + b * (long)p, Xb + b * (long)nstate * M,
                                   M, p, nstate, rho,
                                   Xa + b * (long)nstate * M,
                                   W ? W + b * (long)MM : NULL,
                                   wbar ? wbar + b * (long)M : NULL,
                                   Q, g, lam, V, S, Wl, wb, dX);
            if (info) info[b] = (s < 0) ? 1 : 0;
        }
        free(buf);
    }
    return nt;
}

/* ------------------------------------------------------------------------------------------
 * Grid form (Procedure 1 lines 1-2, Eq.18-19).
 * Every point of a periodic Ny x Nx grid is a local problem whose observations are the V
 * observed variables at the (2 hw + 1)^2 points of the square patch around it:
 *   local row j = v (2hw+1)^2 + (dy+hw)(2hw+1) + (dx+hw),  point (y+dy mod Ny, x+dx mod Nx)
 *   ybar  = mean_m Yf[v][yy][xx][m]                     Eq.18
 *   dY_j  = Yf[v][yy][xx][:] - ybar                     Eq.19
 *   d_j   = yo[v][yy][xx] - ybar                        innovation of Eq.14
 *   r_j   = G(dist) / sigma_o^2, 0 where mask[yy][xx] == 0 (unobserved point, reading G7)
 * with dist = sqrt(dx^2 + dy^2) in grid units and the localisation function G:
 *   loc_kind 0: Gaussian exp(-dist^2 / (2 L^2))                 (BASELINE.json configs)
 *   loc_kind 1: Gaspari-Cohn 5th-order piecewise rational with half-width c = L, zero from
 *               2c on (ref.[21] of the paper; the paper's cutoff 2(p-1) dx is 2c)
 * The local problem itself is analysis_point() above, unchanged.
 */
double oracle_localisation(int loc_kind, double L, double dist)
{
    if (loc_kind == 0) return exp(-(dist * dist) / (2.0 * L * L));
    {
        const double z = dist / L;
        if (z >= 2.0) return 0.0;
        if (z <= 1.0)
            return ((((-0.25 * z + 0.5) * z + 0.625) * z - 5.0 / 3.0) * z) * z + 1.0;
        return (((((1.0 / 12.0) * z - 0.5) * z + 0.625) * z + 5.0 / 3.0) * z - 5.0) * z + 4.0
               - (2.0 / 3.0) / z;
    }
}

int oracle_letkf_analysis_grid(const double* Yf, const double* yo, const unsigned char* mask,
                               const double* Xb, int M, int V, int Ny, int Nx, int nstate,
                               int hw, int loc_kind, double L, double sigma_o, double rho,
                               double* Xa, double* wbar, int* info, int nthreads)
{
    int nt = pick_threads(nthreads);
    const int side = 2 * hw + 1, P2 = side * side, p = V * P2;
    const long npts = (long)Ny * Nx;
    if (M < 1 || V < 1 || Ny < 1 || Nx < 1 || nstate < 1 || hw < 0) return nt;
#pragma omp parallel num_threads(nt)
    {
        size_t MM = (size_t)M * M;
        double* buf = (double*)malloc(sizeof(double) * (4 * MM + 4 * (size_t)M + (size_t)p * M + 2 * (size_t)p));
        double *Q = buf, *Vv = buf + MM, *S = buf + 2 * MM, *Wl = buf + 3 * MM;
        double *g = buf + 4 * MM, *lam = g + M, *wb = lam + M, *dX = wb + M;
        double *Yb = dX + M, *dv = Yb + (size_t)p * M, *rv = dv + p;
        long b;
#pragma omp for schedule(dynamic)
        for (b = 0; b < npts; ++b) {
            const int y = (int)(b / Nx), x = (int)(b % Nx);
            int v, dy, dx, m, sweeps;
            for (v = 0; v < V; ++v)
                for (dy = -hw; dy <= hw; ++dy)
                    for (dx = -hw; dx <= hw; ++dx) {
                        const int j = v * P2 + (dy + hw) * side + (dx + hw);
                        const int yy = ((y + dy) % Ny + Ny) % Ny, xx = ((x + dx) % Nx + Nx) % Nx;
                        const double* src = Yf + (((long)v * Ny + yy) * Nx + xx) * M;
                        double ybar = 0.0;
                        for (m = 0; m < M; ++m) ybar += src[m];
                        ybar /= (double)M;
                        for (m = 0; m < M; ++m) Yb[(long)j * M + m] = src[m] - ybar;
                        dv[j] = yo[((long)v * Ny + yy) * Nx + xx] - ybar;
                        rv[j] = (mask && !mask[(long)yy * Nx + xx])
                                    ? 0.0
                                    : oracle_localisation(loc_kind, L, sqrt((double)(dx * dx + dy * dy)))
                                          / (sigma_o * sigma_o);
                    }
            sweeps = analysis_point(Yb, dv, rv, Xb + b * (long)nstate * M, M, p, nstate, rho,
                                    Xa + b * (long)nstate * M, NULL, wbar ? wbar + b * (long)M : NULL,
                                    Q, g, lam, Vv, S, Wl, wb, dX);
            if (info) info[b] = (sweeps < 0) ? 1 : 0;
        }
        free(buf);
    }
    return nt;
}


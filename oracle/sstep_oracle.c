/*
 * oracle/sstep_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded (see ORC_PAR_FOR below for the one exception), obviously-correct CPU (fp64) implementation of
 * what the s-step PCG hot path of arxiv 2501.03743 computes, written from
 * /root/reference/PAPER.md only.  It shares no code, header, table or helper
 * with the CUDA library in paper_2501_03743_b200/; only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.  Citations are "PAPER.md:<line>" plus the algorithm / equation.
 *
 * Conventions
 *   - CSR: 0-based, int32 rowptr[n+1] / colidx[nnz], double vals[nnz].
 *   - n x s blocks (R, AR, P, AP) are COLUMN-MAJOR with leading dimension n:
 *     column j (0-based) is X + j*n.  This is the paper's P(:, j) notation
 *     (Alg. 4): R = P(:,1:s), AR = P(:,s+1:2s).
 *   - small s x s matrices are ROW-MAJOR: W[i*s + j] = W(i+1, j+1).
 *   - every inner product is accumulated in long double (the oracle is meant
 *     to be the more accurate side at n ~ 3e7); SpMV rows and the block
 *     updates are evaluated in double exactly as the formulas read.
 *   - preconditioner B = diag(A) (reading A14 in DESIGN.md): B^{-1} v is the
 *     multiplication by the precomputed dinv[i] = 1 / a_ii.
 *   - stop test: ||r||_2 < rtol * ||r_0||_2, strict, r the recurrence residual
 *     ("Euclidean norm of the relative residual"; reading A7).
 *   - status: 0 converged, 1 maxit reached, 2 breakdown.
 *
 * Pins: tests/test_oracle_*.py (closed-form Poisson eigenpairs, dense LU,
 * Hilbert inverse, CG <-> s-step iterate identity, A-conjugacy, the classical
 * CG error bound, the paper's 514 iterations, scipy cross-checks).
 */
#define _POSIX_C_SOURCE 199309L /* clock_gettime under -std=c11 (timing instrumentation only) */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>

typedef int32_t i32;
typedef int64_t i64;

#define ORC_SMAX 16

/* All-core timing leg (SURVEY.md 8(d) "Oracle timed beside it", leg 2): the SAME source built a second time with
 * -fopenmp (liboracle_omp.so) runs its row loops and inner products on all host cores.  Without the flag -- the
 * build every pin and every parity test uses -- the two macros below expand to nothing and this file is the
 * single-threaded program it always was, statement for statement.  (With the flag the inner products are summed
 * per thread and then combined, i.e. in another order: that build is for bench.py's cpu_baseline only.) */
#ifdef _OPENMP
#define ORC_PRAGMA(x) _Pragma(#x)
#define ORC_PAR_FOR ORC_PRAGMA(omp parallel for schedule(static))
#define ORC_PAR_SUM(v) ORC_PRAGMA(omp parallel for schedule(static) reduction(+ : v))
#else
#define ORC_PAR_FOR
#define ORC_PAR_SUM(v)
#endif

/* Timing instrumentation for bench.py (no arithmetic): if a log is set, orc_sstep_rr stores the wall clock at the
 * start of its outer loop in tlog[0] and after outer iteration k in tlog[k + 1], so that a caller can time outer
 * iterations without the solver's start-up (dinv, r0). */
static double *orc_tlog = NULL;
static int orc_tlog_cap = 0;
void orc_set_time_log(double *tlog, int cap) { orc_tlog = tlog; orc_tlog_cap = cap; }
static double orc_now(void)
{
    struct timespec ts;
    clock_gettime(CLOCK_MONOTONIC, &ts);
    return (double)ts.tv_sec + 1e-9 * (double)ts.tv_nsec;
}

/* ---------------------------------------------------------------- basics */

/* y = A x  (the operator of Eq. 1) */
void orc_spmv(i64 n, const i32 *rowptr, const i32 *colidx, const double *vals,
              const double *x, double *y)
{
    ORC_PAR_FOR
    for (i64 i = 0; i < n; i++) {
        double acc = 0.0;
        for (i64 k = rowptr[i]; k < rowptr[i + 1]; k++)
            acc += vals[k] * x[colidx[k]];
        y[i] = acc;
    }
}

/* dinv[i] = 1 / a_ii ; returns -1 if a diagonal entry is missing or <= 0 */
int orc_dinv(i64 n, const i32 *rowptr, const i32 *colidx, const double *vals, double *dinv)
{
    for (i64 i = 0; i < n; i++) {
        double d = 0.0;
        int found = 0;
        for (i64 k = rowptr[i]; k < rowptr[i + 1]; k++)
            if (colidx[k] == i) { d = vals[k]; found = 1; }
        if (!found || !(d > 0.0)) return -1;
        dinv[i] = 1.0 / d;
    }
    return 0;
}

static long double ldot(i64 n, const double *a, const double *b)
{
    long double acc = 0.0L;
    ORC_PAR_SUM(acc)
    for (i64 i = 0; i < n; i++) acc += (long double)a[i] * (long double)b[i];
    return acc;
}

double orc_dot(i64 n, const double *a, const double *b) { return (double)ldot(n, a, b); }

/* ---------------------------------------------------------------- MPK
 * Alg. 4: P(:,1) = B^{-1} x, then alternately
 * P(:,s+j) = A P(:,j) and P(:,j+1) = B^{-1} P(:,s+j).  Unrolling pin/pout
 * (1 -> s+1 -> 2 -> s+2 ...) gives R_1 = B^{-1} r, AR_j = A R_j,
 * R_{j+1} = B^{-1} AR_j.
 *
 * basis = 0: the paper's monomial basis (above).
 * basis = 1: scaled-and-shifted Chebyshev basis on [0,2] (DESIGN.md NEXT-1;
 *   motivated by PAPER.md:154-156, 251, 325): with Z = B^{-1}A - I,
 *   R_2 = Z R_1, R_{j+1} = 2 Z R_j - R_{j-1}.  AR_j = A R_j as before.
 */
void orc_mpk(i64 n, const i32 *rowptr, const i32 *colidx, const double *vals,
             const double *dinv, const double *r, int s, int basis, double *R, double *AR)
{
    ORC_PAR_FOR
    for (i64 i = 0; i < n; i++) R[i] = dinv[i] * r[i];
    for (int j = 0; j < s; j++) {
        const double *Rj = R + (i64)j * n;
        double *ARj = AR + (i64)j * n;
        orc_spmv(n, rowptr, colidx, vals, Rj, ARj);
        if (j + 1 < s) {
            double *Rn = R + (i64)(j + 1) * n;
            if (basis == 0) {
                ORC_PAR_FOR
                for (i64 i = 0; i < n; i++) Rn[i] = dinv[i] * ARj[i];
            } else if (j == 0) {
                ORC_PAR_FOR
                for (i64 i = 0; i < n; i++) Rn[i] = dinv[i] * ARj[i] - Rj[i];
            } else {
                const double *Rp = R + (i64)(j - 1) * n;
                ORC_PAR_FOR
                for (i64 i = 0; i < n; i++) Rn[i] = 2.0 * (dinv[i] * ARj[i] - Rj[i]) - Rp[i];
            }
        }
    }
}

/* ---------------------------------------------------------------- Gram
 * The fused block inner products of one outer iteration (north_star; Eq. 3-4,
 * PAPER.md:142-154):
 *   M = R^T AR   (s x s; the paper's moment matrix, M(i,j) = mu^{i+j-1})
 *   C = AP^T R   (s x s; c_i of PAPER.md:148-150, AP = A P_old)
 *   m = R^T r    (s;     right-hand side of Eq. 3 since r is orthogonal to P_old)
 */
void orc_gram(i64 n, int s, const double *R, const double *AR, const double *AP,
              const double *r, double *M, double *C, double *m)
{
    for (int i = 0; i < s; i++) {
        for (int j = 0; j < s; j++) {
            M[i * s + j] = (double)ldot(n, R + (i64)i * n, AR + (i64)j * n);
            C[i * s + j] = AP ? (double)ldot(n, AP + (i64)i * n, R + (i64)j * n) : 0.0;
        }
        m[i] = (double)ldot(n, R + (i64)i * n, r);
    }
}

/* Alg. 5 cvm: vm(1:s) = P(:,1:s)^T r ; vm(s+1:2s) = P(:,1:s)^T P(:,2s) */
void orc_cvm(i64 n, int s, const double *R, const double *AR, const double *r, double *vm)
{
    for (int i = 0; i < s; i++) {
        vm[i] = (double)ldot(n, R + (i64)i * n, r);
        vm[s + i] = (double)ldot(n, R + (i64)i * n, AR + (i64)(s - 1) * n);
    }
}

/* The same 2s moments taken where the matrix-powers kernel produces them (Eq. 4,
 * mu^k = r^T B^{-1} (A B^{-1})^k r):
 *   mu^0 = R_1^T r,  mu^{2j-1} = R_j^T AR_j,  mu^{2j} = R_{j+1}^T AR_j  (j = 1..s; mu^{2s} is not needed).
 * In exact arithmetic vm[k] = mu^k equals orc_cvm's vm (A symmetric); in fp64 the two differ by rounding. */
void orc_cvm_fused(i64 n, int s, const double *R, const double *AR, const double *r, double *vm)
{
    vm[0] = (double)ldot(n, R, r);
    for (int j = 1; j <= s; j++) {
        vm[2 * j - 1] = (double)ldot(n, R + (i64)(j - 1) * n, AR + (i64)(j - 1) * n);
        if (j < s) vm[2 * j] = (double)ldot(n, R + (i64)j * n, AR + (i64)(j - 1) * n);
    }
}

/* ---------------------------------------------------------------- small solves
 * "solve s+1 spd systems of dimension s".  Method (reading A10):
 * Cholesky W = L L^T reading only the lower triangle of W, then forward and
 * back substitution.  Returns 0, or 2 on a non-positive / non-finite pivot.
 */
int orc_chol(int s, const double *W, double *L)
{
    memset(L, 0, sizeof(double) * (size_t)s * s);
    for (int j = 0; j < s; j++) {
        double d = W[j * s + j];
        for (int k = 0; k < j; k++) d -= L[j * s + k] * L[j * s + k];
        if (!(d > 0.0) || !isfinite(d)) return 2;
        double ljj = sqrt(d);
        L[j * s + j] = ljj;
        for (int i = j + 1; i < s; i++) {
            double v = W[i * s + j];
            for (int k = 0; k < j; k++) v -= L[i * s + k] * L[j * s + k];
            L[i * s + j] = v / ljj;
        }
    }
    return 0;
}

/* X = W^{-1} B for nrhs right-hand sides; B, X are s x nrhs row-major; L from orc_chol */
void orc_chol_solve(int s, const double *L, int nrhs, const double *B, double *X)
{
    for (int c = 0; c < nrhs; c++) {
        double y[ORC_SMAX];
        for (int i = 0; i < s; i++) {
            double v = B[i * nrhs + c];
            for (int k = 0; k < i; k++) v -= L[i * s + k] * y[k];
            y[i] = v / L[i * s + i];
        }
        for (int i = s - 1; i >= 0; i--) {
            double v = y[i];
            for (int k = i + 1; k < s; k++) v -= L[k * s + i] * X[k * nrhs + c];
            X[i * nrhs + c] = v / L[i * s + i];
        }
    }
}

/* Gram-form scalar work (Alg. 3 l.7-16 with SW written on the Gram blocks):
 *   first:  beta = 0, W = M                      (Alg. 3 l.8-14)
 *   else:   W_prev beta + C = 0
 *           W = M + C^T beta                     (= M_i - c_i beta_{i-1})
 *   alpha:  W alpha = m                          (Eq. 3)
 */
int orc_small_solve(int s, int first, const double *M, const double *C, const double *m,
                    const double *Wprev, double *beta, double *alpha, double *W)
{
    double L[ORC_SMAX * ORC_SMAX], negC[ORC_SMAX * ORC_SMAX];
    if (first) {
        for (int i = 0; i < s * s; i++) { beta[i] = 0.0; W[i] = M[i]; }
    } else {
        int st = orc_chol(s, Wprev, L);
        if (st) return st;
        for (int i = 0; i < s * s; i++) negC[i] = -C[i];
        orc_chol_solve(s, L, s, negC, beta);
        for (int i = 0; i < s; i++)
            for (int j = 0; j < s; j++) {
                double v = M[i * s + j];
                for (int l = 0; l < s; l++) v += C[l * s + i] * beta[l * s + j];
                W[i * s + j] = v;
            }
    }
    int st = orc_chol(s, W, L);
    if (st) return st;
    orc_chol_solve(s, L, 1, m, alpha);
    for (int i = 0; i < s; i++) if (!isfinite(alpha[i])) return 2;
    return 0;
}

/* Alg. 6 SW(alpha, beta, W, vm, s), paper-literal moment form.
 * In: vm (2s moments of the new residual), alpha and W of the PREVIOUS outer
 * iteration (reading A3).  Out: beta, and alpha, W overwritten.
 * Readings: A2 - l.5 reads rhs(s-1+i) += rhs(s-1+j) * alpha(s-i+j);
 * A1 - the fill of b1 at l.9-13 runs over all j = 1..s (full Hankel), not
 * j = 1..i-1 as printed.
 */
int orc_sw(int s, const double *vm, double *alpha, double *beta, double *W)
{
    double rhs[2 * ORC_SMAX], b1[ORC_SMAX * ORC_SMAX], L[ORC_SMAX * ORC_SMAX];
    double Mh[ORC_SMAX * ORC_SMAX];
    if (alpha[s - 1] == 0.0 || !isfinite(alpha[s - 1])) return 2;
    for (int i = 0; i < 2 * s - 1; i++) rhs[i] = 0.0;              /* l.1  */
    for (int i = 1; i <= s; i++) {                                  /* l.2  */
        double t = vm[i - 1];                                       /* l.3  */
        for (int j = 1; j <= i - 1; j++)                            /* l.4  */
            t += rhs[s - 1 + j - 1] * alpha[s - i + j - 1];         /* l.5  */
        rhs[s - 1 + i - 1] = -t / alpha[s - 1];                     /* l.7  */
    }
    for (int i = 1; i <= s; i++)                                    /* l.9  */
        for (int j = 1; j <= s; j++)                                /* l.10 (A1) */
            b1[(i - 1) * s + (j - 1)] = -rhs[i + j - 1 - 1];        /* l.11 */
    int st = orc_chol(s, W, L);
    if (st) return st;
    orc_chol_solve(s, L, s, b1, beta);                              /* l.14 */
    for (int i = 1; i <= s; i++)                                    /* l.15-19 */
        for (int j = 1; j <= s; j++)
            Mh[(i - 1) * s + (j - 1)] = vm[i + j - 1];
    for (int i = 0; i < s; i++)                                     /* l.20 */
        for (int j = 0; j < s; j++) {
            double v = Mh[i * s + j];
            for (int l = 0; l < s; l++) v -= b1[i * s + l] * beta[l * s + j];
            W[i * s + j] = v;
        }
    st = orc_chol(s, W, L);
    if (st) return st;
    orc_chol_solve(s, L, 1, vm, alpha);                             /* l.21 */
    for (int i = 0; i < s; i++) if (!isfinite(alpha[i])) return 2;
    return 0;
}

/* ---------------------------------------------------------------- block updates
 * Alg. 3 l.17-21, in place:
 *   P  <- R  + P  beta      x <- x + P  alpha
 *   AP <- AR + AP beta      r <- r - AP alpha
 * R/AR are this iteration's MPK output, P/AP the previous directions (the
 * paper's P2/P1 ping-pong is double buffering of exactly this).
 */
void orc_update(i64 n, int s, const double *R, const double *AR, double *P, double *AP,
                double *x, double *r, const double *beta, const double *alpha)
{
    ORC_PAR_FOR
    for (i64 i = 0; i < n; i++) {
        double pn[ORC_SMAX], apn[ORC_SMAX];
        for (int j = 0; j < s; j++) {
            double p = R[(i64)j * n + i], ap = AR[(i64)j * n + i];
            for (int l = 0; l < s; l++) {
                p += P[(i64)l * n + i] * beta[l * s + j];
                ap += AP[(i64)l * n + i] * beta[l * s + j];
            }
            pn[j] = p; apn[j] = ap;
        }
        double xi = x[i], ri = r[i];
        for (int j = 0; j < s; j++) {
            P[(i64)j * n + i] = pn[j];
            AP[(i64)j * n + i] = apn[j];
            xi += pn[j] * alpha[j];
            ri -= apn[j] * alpha[j];
        }
        x[i] = xi; r[i] = ri;
    }
}

/* ---------------------------------------------------------------- solvers
 * Common outputs: x (n), *iters, *relres (= ||r||/||r0|| at exit),
 * hist[k] = ||r_{k+1}||/||r_0|| after iteration k (NULL or >= maxit entries),
 * xhist: NULL or n*xhist_cap doubles, iterate after iteration k at xhist+k*n.
 */
static void init_residual(i64 n, const i32 *rp, const i32 *ci, const double *v,
                          const double *b, const double *x0, double *x, double *r)
{
    if (x0) {
        memcpy(x, x0, sizeof(double) * (size_t)n);
        orc_spmv(n, rp, ci, v, x, r);
        for (i64 i = 0; i < n; i++) r[i] = b[i] - r[i];
    } else {
        memset(x, 0, sizeof(double) * (size_t)n);
        memcpy(r, b, sizeof(double) * (size_t)n);
    }
}

/* Alg. 1 PCG-HS */
int orc_pcg(i64 n, const i32 *rp, const i32 *ci, const double *v, const double *b,
            const double *x0, double rtol, int maxit, double *x, int *iters, double *relres,
            double *hist, double *xhist, int xhist_cap)
{
    double *r = malloc(sizeof(double) * n), *u = malloc(sizeof(double) * n);
    double *p = malloc(sizeof(double) * n), *sk = malloc(sizeof(double) * n);
    double *dinv = malloc(sizeof(double) * n);
    int status = 1;
    *iters = 0;
    if (orc_dinv(n, rp, ci, v, dinv)) { status = -1; goto done; }
    init_residual(n, rp, ci, v, b, x0, x, r);                         /* l.1 */
    double nr0 = sqrt((double)ldot(n, r, r));
    *relres = 1.0;
    if (nr0 == 0.0) { status = 0; *relres = 0.0; goto done; }
    for (i64 i = 0; i < n; i++) { u[i] = dinv[i] * r[i]; p[i] = u[i]; } /* l.2-3 */
    double ur = (double)ldot(n, u, r);
    for (int k = 0; k < maxit; k++) {                                  /* l.4 */
        orc_spmv(n, rp, ci, v, p, sk);                                 /* s_k = A p_k */
        double ps = (double)ldot(n, p, sk);
        if (!(ps > 0.0) || !isfinite(ps)) { status = 2; break; }
        double alpha = ur / ps;                                        /* alpha_k */
        for (i64 i = 0; i < n; i++) { x[i] += alpha * p[i]; r[i] -= alpha * sk[i]; }
        for (i64 i = 0; i < n; i++) u[i] = dinv[i] * r[i];             /* u_{k+1} */
        double ur_new = (double)ldot(n, u, r);
        double beta = ur_new / ur;                                     /* beta_k */
        for (i64 i = 0; i < n; i++) p[i] = u[i] + beta * p[i];
        ur = ur_new;
        double nr = sqrt((double)ldot(n, r, r));
        *iters = k + 1;
        *relres = nr / nr0;
        if (hist) hist[k] = *relres;
        if (xhist && k < xhist_cap) memcpy(xhist + (i64)k * n, x, sizeof(double) * n);
        if (nr < rtol * nr0) { status = 0; break; }                    /* l.11-13 */
    }
done:
    free(r); free(u); free(p); free(sk); free(dinv);
    return status;
}

/* Alg. 2 PFCG-NN.  One "iteration" = one SpMV step: the
 * start-up l.1-7 is iteration 1, each pass of the loop one more.  The stop test
 * is also applied after the start-up step (the printed loop only tests inside). */
int orc_pfcg(i64 n, const i32 *rp, const i32 *ci, const double *v, const double *b,
             const double *x0, double rtol, int maxit, double *x, int *iters, double *relres,
             double *hist, double *xhist, int xhist_cap)
{
    double *r = malloc(sizeof(double) * n), *u = malloc(sizeof(double) * n);
    double *p = malloc(sizeof(double) * n), *sv = malloc(sizeof(double) * n);
    double *w = malloc(sizeof(double) * n), *dinv = malloc(sizeof(double) * n);
    int status = 1;
    *iters = 0;
    if (orc_dinv(n, rp, ci, v, dinv)) { status = -1; goto done; }
    init_residual(n, rp, ci, v, b, x0, x, r);                          /* l.1 */
    double nr0 = sqrt((double)ldot(n, r, r));
    *relres = 1.0;
    if (nr0 == 0.0) { status = 0; *relres = 0.0; goto done; }
    double rho_prev = 0.0;
    for (int k = 0; k < maxit; k++) {
        for (i64 i = 0; i < n; i++) u[i] = dinv[i] * r[i];             /* u_k = B^{-1} r_k */
        orc_spmv(n, rp, ci, v, u, w);                                  /* w_k = A u_k */
        double alpha = (double)ldot(n, u, r);                          /* l.11 */
        double beta = (double)ldot(n, u, w);                           /* l.12 */
        double gamma = (k == 0) ? 0.0 : (double)ldot(n, u, sv);        /* l.13 */
        double rho = (k == 0) ? beta : beta - gamma * gamma / rho_prev; /* l.5 / l.14 */
        if (!(rho > 0.0) || !isfinite(rho)) { status = 2; break; }
        if (k == 0) {
            for (i64 i = 0; i < n; i++) { p[i] = u[i]; sv[i] = w[i]; }  /* l.2-3 */
        } else {
            double g = gamma / rho_prev;
            for (i64 i = 0; i < n; i++) { p[i] = u[i] - g * p[i]; sv[i] = w[i] - g * sv[i]; } /* l.15,17 */
        }
        double a = alpha / rho;
        for (i64 i = 0; i < n; i++) { x[i] += a * p[i]; r[i] -= a * sv[i]; } /* l.16,18 */
        rho_prev = rho;
        double nr = sqrt((double)ldot(n, r, r));
        *iters = k + 1;
        *relres = nr / nr0;
        if (hist) hist[k] = *relres;
        if (xhist && k < xhist_cap) memcpy(xhist + (i64)k * n, x, sizeof(double) * n);
        if (nr < rtol * nr0) { status = 0; break; }
    }
done:
    free(r); free(u); free(p); free(sv); free(w); free(dinv);
    return status;
}

/* Alg. 3 PCGs, outer loop.
 *   form = 0: Gram form (O2 in DESIGN.md; the CUDA path's twin): orc_gram + orc_small_solve
 *   form = 1: paper-literal moment form (O3): orc_cvm (Alg. 5) + orc_sw (Alg. 6)
 * maxit counts OUTER iterations (reading A9); *iters = outer iterations done.
 */
/* replace_every = R > 0: residual replacement (related work; reading A22 of DESIGN.md).  After the block
 * update of every R-th outer iteration -- unless the recurrence residual has just passed the stop test -- r is
 * overwritten by the true residual b - A x (one extra SpMV), the directions P, AP are kept, and the stop test is taken
 * again on the replaced residual; hist[k] then holds the replaced value.  R = 0: never (Alg. 3 as printed). */
int orc_sstep_rr(i64 n, const i32 *rp, const i32 *ci, const double *v, const double *b,
                 const double *x0, int s, int form, int basis, int replace_every, double rtol, int maxit, double *x,
                 int *iters, double *relres, double *hist, double *xhist, int xhist_cap)
{
    if (s < 1 || s > ORC_SMAX) return -1;
    size_t blk = sizeof(double) * (size_t)n * s;
    double *r = malloc(sizeof(double) * n), *dinv = malloc(sizeof(double) * n);
    double *R = malloc(blk), *AR = malloc(blk), *P = calloc((size_t)n * s, sizeof(double));
    double *AP = calloc((size_t)n * s, sizeof(double));
    double M[ORC_SMAX * ORC_SMAX], C[ORC_SMAX * ORC_SMAX], m[ORC_SMAX], vm[2 * ORC_SMAX];
    double W[ORC_SMAX * ORC_SMAX], Wn[ORC_SMAX * ORC_SMAX], beta[ORC_SMAX * ORC_SMAX], alpha[ORC_SMAX];
    int status = 1;
    *iters = 0;
    if (orc_dinv(n, rp, ci, v, dinv)) { status = -1; goto done; }
    init_residual(n, rp, ci, v, b, x0, x, r);                          /* l.1 */
    double nr0 = sqrt((double)ldot(n, r, r));
    *relres = 1.0;
    if (nr0 == 0.0) { status = 0; *relres = 0.0; goto done; }
    if (orc_tlog && orc_tlog_cap > 0) orc_tlog[0] = orc_now();
    for (int k = 0; k < maxit; k++) {                                  /* l.3 */
        orc_mpk(n, rp, ci, v, dinv, r, s, basis, R, AR);               /* l.5 / l.23 */
        int st;
        if (form == 0) {
            orc_gram(n, s, R, AR, k ? AP : NULL, r, M, C, m);
            st = orc_small_solve(s, k == 0, M, C, m, W, beta, alpha, Wn);
            memcpy(W, Wn, sizeof(double) * s * s);
        } else {
            if (form == 2) orc_cvm_fused(n, s, R, AR, r, vm);          /* moments from the MPK epilogues */
            else orc_cvm(n, s, R, AR, r, vm);                          /* l.6 / l.24 */
            if (k == 0) {                                              /* l.7-14 */
                for (int i = 1; i <= s; i++)
                    for (int j = 1; j <= s; j++) W[(i - 1) * s + (j - 1)] = vm[i + j - 1];
                for (int i = 0; i < s * s; i++) beta[i] = 0.0;
                double L[ORC_SMAX * ORC_SMAX];
                st = orc_chol(s, W, L);
                if (!st) orc_chol_solve(s, L, 1, vm, alpha);
            } else {
                st = orc_sw(s, vm, alpha, beta, W);                    /* l.16 / l.25 */
            }
        }
        if (st) { status = 2; break; }
        orc_update(n, s, R, AR, P, AP, x, r, beta, alpha);             /* l.17-21 / l.26-30 */
        double nr = sqrt((double)ldot(n, r, r));
        *iters = k + 1;
        *relres = nr / nr0;
        if (hist) hist[k] = *relres;
        if (xhist && k < xhist_cap) memcpy(xhist + (i64)k * n, x, sizeof(double) * n);
        if (orc_tlog && k + 1 < orc_tlog_cap) orc_tlog[k + 1] = orc_now();
        if (!isfinite(nr)) { status = 2; break; }
        if (nr < rtol * nr0) { status = 0; break; }                    /* l.31-33 */
        if (replace_every > 0 && (k + 1) % replace_every == 0) {
            orc_spmv(n, rp, ci, v, x, R);                              /* R(:,1) is scratch here: the next MPK rewrites it */
            for (i64 i = 0; i < n; i++) r[i] = b[i] - R[i];
            nr = sqrt((double)ldot(n, r, r));
            *relres = nr / nr0;
            if (hist) hist[k] = *relres;
            if (!isfinite(nr)) { status = 2; break; }
            if (nr < rtol * nr0) { status = 0; break; }
        }
    }
done:
    free(r); free(dinv); free(R); free(AR); free(P); free(AP);
    return status;
}

int orc_sstep(i64 n, const i32 *rp, const i32 *ci, const double *v, const double *b,
              const double *x0, int s, int form, int basis, double rtol, int maxit, double *x,
              int *iters, double *relres, double *hist, double *xhist, int xhist_cap)
{
    return orc_sstep_rr(n, rp, ci, v, b, x0, s, form, basis, 0, rtol, maxit, x, iters, relres, hist, xhist, xhist_cap);
}

/*
 * sstep_cg.h -- C ABI of the B200-native s-step preconditioned CG hot path
 * (Chronopoulos-Gear s-step PCG as described in arxiv 2501.03743).
 *
 * Problem statement: solve A x = b, A symmetric positive definite, with an spd
 * preconditioner B (Eq. 1).  Solver signature
 * PCGs(A, b, B, x0, s, rtol, kmax) (Alg. 3); B = diag(A) here.
 *
 * One OUTER iteration (Alg. 3 l.5-21) is, on the device, in one CUDA graph:
 *   a1  matrix-powers kernel, Alg. 4: R_1 = D^-1 r and, for
 *       j = 1..s, AR_j = A R_j, R_{j+1} = D^-1 AR_j  (s Jacobi-fused CSR SpMVs)
 *   a2  fused block inner products in one pass (Eq. 3-4, PAPER.md:142-154;
 *       generalises Alg. 5): M = R^T AR, C = AP^T R, m = R^T r
 *   a3  on-device s x s solves: W_prev beta = -C,
 *       W = M + C^T beta, W alpha = m   (Cholesky, one warp)
 *   a4  fused block updates (Alg. 3 l.17-21): P <- R + P beta, AP <- AR + AP beta,
 *       x <- x + P alpha, r <- r - AP alpha, plus R_1 <- D^-1 r and ||r||^2
 *   a5  stop test ||r||_2 < rtol * ||r_0||_2 (Alg. 3 l.31-33)
 *
 * General rules
 *   - All functions return an int: 0 = success / converged, > 0 = solver
 *     outcome (see SSTEP_CG_* below), < 0 = invalid argument or CUDA error
 *     (text via sstep_cg_last_error).  No exceptions, no global state.
 *   - Pointers are DEVICE pointers unless the name ends in _host.  fp64 values,
 *     int32 indices.  All work is enqueued on the stream given at create();
 *     functions that return results to the host synchronise that stream.
 *   - CSR: 0-based, rowptr[n+1], colidx[nnz], vals[nnz]; every row holds its
 *     diagonal entry exactly once and it is > 0 (checked at setup).  Column order inside a
 *     row is free; other duplicated (row, column) entries are summed.
 *     The three arrays are BORROWED: the caller keeps them alive and unchanged
 *     until sstep_cg_destroy or the next sstep_cg_setup.
 *   - n x s blocks in the test hooks use two layouts:
 *       column-major ("cm"): element (i, j) at X[j*n + i]   -- R, AR
 *       interleaved  ("il"): element (i, j) at X[i*s + j]   -- P, AP
 *     small s x s matrices are row-major: W[i*s + j].
 *   - There is no CPU fallback: every entry point fails with
 *     SSTEP_CG_ERR_CUDA if no sm_100 device is usable.
 */
#ifndef SSTEP_CG_H
#define SSTEP_CG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SSTEP_CG_SMAX 16           /* largest supported block size s */

/* solver outcomes (return value of solve / field status) */
#define SSTEP_CG_CONVERGED 0       /* ||r|| < rtol ||r0||                                   */
#define SSTEP_CG_MAXIT 1           /* "did not converge within kmax iterations"; x valid */
#define SSTEP_CG_BREAKDOWN 2       /* numerical breakdown.  Non-positive / non-finite Cholesky pivot or non-finite alpha
                                    * (detected BEFORE the block update, which is then skipped): x = the last good
                                    * iterate.  Non-finite ||r||^2 after a block update (overflow inside it): x, r, P, AP
                                    * already hold that update and may be non-finite -- restart from your own x0. */
#define SSTEP_CG_RUNNING (-1)      /* only in sstep_cg_solve_peek's out->status: the stop test has not fired yet */
/* errors */
#define SSTEP_CG_ERR_ARG (-1)
#define SSTEP_CG_ERR_CUDA (-2)
#define SSTEP_CG_ERR_STATE (-3)    /* call order violated (e.g. solve before setup) */
#define SSTEP_CG_ERR_MATRIX (-4)   /* rowptr inconsistent, missing or non-positive diagonal */

/* basis of the matrix-powers kernel */
#define SSTEP_CG_BASIS_MONOMIAL 0  /* the paper's basis, Alg. 4 */
#define SSTEP_CG_BASIS_CHEBYSHEV 1 /* Chebyshev on [0,2] for D^-1 A (NEXT-1) */

typedef struct sstep_cg sstep_cg_t;

typedef struct sstep_cg_result {
    int32_t status;          /* SSTEP_CG_CONVERGED / MAXIT / BREAKDOWN */
    int32_t outer_iters;     /* outer iterations executed */
    int64_t cg_equiv_iters;  /* s * outer_iters ("one iteration of PCGs corresponds to s iterations") */
    double relres;           /* ||r||_2 / ||r_0||_2, recurrence residual, at exit */
    double r0_norm;          /* ||r_0||_2 */
    double solve_seconds;    /* host wall time of the call (informative) */
    int64_t kernel_launches; /* kernels this call enqueued (graph nodes x replays + init) */
} sstep_cg_result;

/* Create a solver bound to CUDA device `device` and to `cuda_stream` (a
 * cudaStream_t passed as void*, borrowed; NULL = the legacy default stream).
 * Allocates nothing problem-sized. */
int sstep_cg_create(sstep_cg_t **handle, int device, void *cuda_stream);

/* Bind a matrix and a block size.  Validates (n > 0, 1 <= s <= SSTEP_CG_SMAX,
 * rowptr[0] = 0, rowptr[n] = nnz, diagonal present and > 0), computes
 * dinv = 1/a_ii, picks the SpMV variant from the row-length statistics,
 * allocates the workspaces (R, AR, P, AP: n x s each; x, r, dinv: n) and
 * captures the outer iteration into a CUDA graph.  Re-callable. */
int sstep_cg_setup(sstep_cg_t *handle, int64_t n, int64_t nnz, const int32_t *rowptr,
                   const int32_t *colidx, const double *vals, int s);

/* Options, to be set between create and setup (unknown key -> ERR_ARG):
 *   "basis"        0 monomial (default) | 1 chebyshev
 *   "spmv_variant" 0 auto (default) | 1 force the generic vector-per-row kernel | 2 force the bulk-staged kernel with
 *                  per-warp rings | 3 force the CTA-pipelined bulk-staged kernel (thread-per-row matrices; auto picks it
 *                  there: few large bulk copies in flight per SM instead of many small ones)
 *   "spmv_cta_depth" 2 (default) | 3 | 4 stages of the CTA-pipelined SpMV's ring; "spmv_cta_per_sm" 2 | 3 (default) CTAs per SM
 *   "lanes"        0 auto | 1,2,4,8,16,32 lanes per row
 *   "spmv_depth"   2 (default) | 3 | 4 slots of the bulk-staged SpMV's per-warp shared-memory ring
 *   "block_variant" 0 auto (default: Gram/update through the TMA tile pipeline for s >= 5, register kernels below)
 *                  | 1 force the register kernels | 2 force the tile pipeline
 *   "form"         0 (default) Gram form: fused block inner products M, C, m + Cholesky solves (a2, a3)
 *                  | 1 moment form (paper-literal Alg. 5 + Alg. 6): the 2s moments are accumulated
 *                    in the SpMV epilogues (mu^0 in the update kernel), a one-block kernel runs the scalar work `SW`;
 *                    no Gram pass over R, AR, AP, r.  Monomial basis only; less robust (Hankel assumption, division
 *                    by alpha_prev(s)).
 *   "resident"     0 auto (default) | 1 off | 2 force.  The resident path runs the WHOLE loop of
 *                  Alg. 3 in one cooperative launch: every CTA keeps its rows of the CSR arrays and of R, AR, P, AP, x, r
 *                  in shared memory for the whole solve; no kernel boundary inside the loop (see "resident_sync").  Auto picks it when every CTA's share fits shared memory (n up to a few 10^5 rows; the
 *                  launch-bound regime, e.g. config 1), s <= 4 and form = 0; same arithmetic per row, same status codes.
 *   "resident_sync" 0 (default) | 1.  How the CTAs of the resident path exchange data.  0: flag-in-data -- every published
 *                  double (R_j for the neighbours' gathers, the Gram partials, their sums) travels as two 64-bit words that
 *                  carry a generation tag, readers poll for the tag; no grid barrier, no fence; the sums are formed by one
 *                  CTA per entry and pushed into per-CTA inboxes; ||r||^2 rides in the next iteration's exchange, so the stop
 *                  test is taken one matrix-powers kernel late (same x, same iteration count).  1: round 1's s + 1 grid
 *                  barriers per outer iteration.  Same arithmetic, same bits; config 1: 8.0 us against 11.4 us per iteration.
 *   "reorder"      0 auto (default) | 1 off | 2 force.  Setup-time symmetric reordering A' = Pi A Pi^T for gather locality
 *                  (Cuthill-McKee numbering computed on the device, csrc/reorder.cuh); the solver then owns a permuted
 *                  copy of the CSR arrays, permutes b and x0 on the way in and x on the way out.  In exact arithmetic
 *                  every iterate is unchanged (the Jacobi preconditioner commutes with Pi); in fp64 only the order of
 *                  the Gram sums changes.  Auto: n >= 2^23 rows (the gathered vector cannot live in L2) and more than a
 *                  quarter of the entries further than 2^20 rows from the diagonal (e.g. config 5's randomly permuted
 *                  rows, where every 8-byte gather otherwise costs a 64-byte DRAM access).
 *   "replace_every" 0 never (default, Alg. 3 as printed) | R > 0: residual replacement: after the block update
 *                  of every R-th outer iteration -- unless the recurrence residual has just passed the stop test -- r is
 *                  overwritten by the true residual b - A x (one extra SpMV + one pass), R_1 = D^-1 r and ||r||^2 follow,
 *                  the directions P, AP are kept and the stop test is taken again.  Gram form only; such solves run on
 *                  the graph path; b must stay valid until solve_end.
 *   "method"       0 (default) the s-step PCG of Alg. 3 | 1 the textbook PCG of Alg. 1 (PCG-HS) as its own
 *                  kernel sequence (SpMV with the p^T A p partials, fused x / r / u update with both reductions and the
 *                  stop test, direction update): the classical two-reduction comparator.  Needs s = 1 at setup;
 *                  "outer iterations" are then CG iterations.  (The paper's one-reduction baseline "fcg", Alg. 2, is
 *                  method 0 with s = 1.)
 *   "pdl"          1 (default) | 0.  Programmatic dependent launch: the kernels of one outer iteration (a1 x s, a2 + a3, a4)
 *                  carry the programmatic-stream-serialization attribute, captured as programmatic edges of the graph, so
 *                  the next kernel's blocks become resident while the current one drains (the SpMV also stages its first
 *                  CSR tiles there); each kernel reads or writes solver data only behind `griddepcontrol.wait`, i.e. after
 *                  its predecessor has completed -- results are bitwise those of pdl = 0.  Falls back to 0 by itself if
 *                  the driver cannot capture such a graph (get_info "pdl" tells).
 *   "use_graph"    1 (default) | 0 launch kernels directly (debugging) */
int sstep_cg_set_option(sstep_cg_t *handle, const char *key, int64_t value);
int sstep_cg_get_info(sstep_cg_t *handle, const char *key, int64_t *value);

/* Solve A x = b from x0 (NULL = zeros).  `x` is caller-owned output and may
 * alias x0.  Runs until ||r||_2 < rtol ||r_0||_2 (strict; recurrence
 * residual), `maxit` OUTER iterations, or breakdown.  Returns the status that
 * is also stored in out->status (out may be NULL). */
int sstep_cg_solve(sstep_cg_t *handle, const double *b, const double *x0, double *x,
                   double rtol, int maxit, sstep_cg_result *out);

/* The same solve in three steps, for timing exactly k outer iterations:
 *   begin   : r = b - A x0, R_1 = D^-1 r, P = AP = 0, W_prev = I, k = 0 (asynchronous)
 *   iterate : enqueue `k_outer` replays of the outer-iteration graph (asynchronous, no
 *             host synchronisation; iterations after convergence/breakdown exit early on a device flag)
 *   end     : copy x out, synchronise, fill `out` */
int sstep_cg_solve_begin(sstep_cg_t *handle, const double *b, const double *x0, double rtol);
int sstep_cg_iterate(sstep_cg_t *handle, int k_outer);
int sstep_cg_solve_end(sstep_cg_t *handle, double *x, sstep_cg_result *out);
/* Between solve_begin and solve_end: synchronise the stream and report where the solve stands (outer_iters, relres of
 * the recurrence residual after the last completed outer iteration -- the history of Alg. 3 l.31-33 when called after
 * every sstep_cg_iterate(h, 1) -- and status = SSTEP_CG_RUNNING / CONVERGED / BREAKDOWN).  The solve goes on. */
int sstep_cg_solve_peek(sstep_cg_t *handle, sstep_cg_result *out);

/* End-to-end convenience with HOST buffers: uploads CSR, b, x0 (NULL = zeros),
 * runs setup + solve on a private device copy, downloads x.  This is the call
 * bench.py's `e2e` number times.  The device copy belongs to the handle: its storage is
 * kept for the next call with the same n and nnz (contents are uploaded afresh every call),
 * replaced when the sizes change and released by sstep_cg_destroy. */
int sstep_cg_solve_host(sstep_cg_t *handle, int64_t n, int64_t nnz, const int32_t *rowptr_host,
                        const int32_t *colidx_host, const double *vals_host, const double *b_host,
                        const double *x0_host, double *x_host, int s, double rtol, int maxit,
                        sstep_cg_result *out);

/* Measurement aid (bench.py's `roofline` object).  Between solve_begin and solve_end: run `reps` outer
 * iterations on the live solve state with the kernels launched one by one (no graph) and a CUDA event pair
 * around every launch on the solver's stream.  ms_host[0] = summed device milliseconds of the s*reps SpMV
 * launches, ms_host[1] = of the reps Gram+solve launches, ms_host[2] = of the reps update launches.
 * Synchronises the stream.  The iterations count as real ones (x, r, k advance). */
int sstep_cg_profile_outer(sstep_cg_t *handle, int reps, double *ms_host);

/* Measurement aid (bench.py's read-side peak): stream a private zero-filled buffer of `bytes` bytes (>= 1 MiB, rounded
 * down to 8 KiB) `passes` times inside one launch with hand-written kernels that use the hot path's own load
 * instructions, `reps` timed launches after one warm-up (CUDA events on the solver's stream):
 *   variant 0  128-bit ld.global.nc.L1::no_allocate reads     (Gram / update kernels' loads)
 *   variant 1  cp.async.bulk reads, 24 warps x 2 x 4 KiB per SM: 48 bulk copies in flight per SM
 *   variant 3  cp.async.bulk reads, 24 warps x 4 x 2 KiB: 96 in flight (the shape of round 1's per-warp SpMV rings)
 *   variant 4  cp.async.bulk reads, 12 warps x 2 x 8 KiB: 24 in flight
 *   variant 5  cp.async.bulk reads, 16 warps x 2 x 4 KiB: 32 in flight (the bulk path is at full speed up to ~32)
 *   variant 2  128-bit copy; read + written bytes both counted (comparable with MEASURED_PEAKS.json hbm_gbs)
 * gbs_out_host[0] = best, [1] = mean GB/s.  bytes >> L2 with passes = 1 gives the HBM figure; a buffer that fits L2
 * with passes > 1 gives the L2-hit bandwidth.  Not allowed during a solve. */
int sstep_cg_measure_bandwidth(sstep_cg_t *handle, int variant, int64_t bytes, int passes, int reps, double *gbs_out_host);

int sstep_cg_destroy(sstep_cg_t *handle);

/* Text of the last failure on this handle ("" if none).  Never NULL. */
const char *sstep_cg_last_error(sstep_cg_t *handle);

/* The row numbering the solver works in: perm_out[i'] (device, n int32) = the caller's index of the solver's row i'
 * (the identity unless setup reordered the matrix, option "reorder").  sstep_cg_solve / solve_begin / solve_end /
 * solve_host take and return vectors in the CALLER's numbering; the test hooks below and sstep_cg_test_read_state
 * work in the SOLVER's numbering (v'[i'] = v[perm[i']]). */
int sstep_cg_get_permutation(sstep_cg_t *handle, int32_t *perm_out);

/* ---- test hooks: run exactly the production kernels on caller-supplied device buffers ---- */

/* Copy one internal array of the current solve state to `out` (device, `count` doubles), after solve_begin / iterate:
 * "R", "AR" (n*s, column-major: the basis blocks of the last MPK; R(:,1) already holds D^-1 r of the NEXT iteration),
 * "P", "AP" (n*s, interleaved), "x", "r" (n), "M", "C", "W", "beta" (s*s, row-major), "m", "alpha" (s).
 * Lets the parity tests check every stage of an outer iteration of the graph AND the resident path on identical
 * inputs (the state before the iteration).  Synchronises the stream. */
int sstep_cg_test_read_state(sstep_cg_t *handle, const char *name, double *out, int64_t count);

/* a1, one SpMV of the matrix-powers kernel: y = A x; if yjac != NULL also yjac = D^-1 y. */
int sstep_cg_test_spmv(sstep_cg_t *handle, const double *x, double *y, double *yjac);
/* a1, Alg. 4: R(:,1) = D^-1 r, then the s fused SpMVs.  R, AR column-major n x s. */
int sstep_cg_test_mpk(sstep_cg_t *handle, const double *r, double *R_cm, double *AR_cm);
/* moment form (option form = 1): Alg. 4 as above and the 2s moments vm[k] = mu^k the SpMV epilogues leave
 * (mu^0 = R_1^T r, mu^{2j-1} = R_j^T AR_j, mu^{2j} = R_{j+1}^T AR_j).  vm: 2s doubles, device. */
int sstep_cg_test_mpk_moments(sstep_cg_t *handle, const double *r, double *R_cm, double *AR_cm, double *vm);
/* Alg. 6 `SW`: from the 2s moments vm and (first == 0) the previous alpha, W (passed in alpha / W, overwritten):
 * beta, alpha, W; first != 0: W = M, beta = 0, alpha = W^-1 vm(1:s).  status_out[0] = 0 or SSTEP_CG_BREAKDOWN. */
int sstep_cg_test_sw(sstep_cg_t *handle, const double *vm, int first, double *beta, double *alpha, double *W,
                     int32_t *status_out);
/* a2: M = R^T AR, C = AP^T R, m = R^T r.  R, AR column-major; AP interleaved; M, C (s*s), m (s) device outputs. */
int sstep_cg_test_gram(sstep_cg_t *handle, const double *R_cm, const double *AR_cm, const double *AP_il,
                       const double *r, double *M, double *C, double *m);
/* a3: beta = -Wprev^-1 C, W = M + C^T beta, alpha = W^-1 m; status_out[0] = 0 or SSTEP_CG_BREAKDOWN. */
int sstep_cg_test_small_solve(sstep_cg_t *handle, const double *M, const double *C, const double *m,
                              const double *Wprev, double *beta, double *alpha, double *W, int32_t *status_out);
/* a3 as the solver loop runs it: the Cholesky factor of the previous W is carried over instead of recomputed
 * (Lprev: s*s row-major, lower triangle, zeros above); Lout = the factor of the new W.  Same bits as the call above
 * with Wprev = Lprev Lprev^T's source matrix, because that call computes exactly this factor first. */
int sstep_cg_test_small_solve_carried(sstep_cg_t *handle, const double *M, const double *C, const double *m,
                                      const double *Lprev, double *beta, double *alpha, double *W, double *Lout,
                                      int32_t *status_out);
/* The division inside the register version of a3 (resident path, s <= 2; csrc/small_solve.cuh): the IEEE quotient a / b
 * computed as "reciprocal of b prepared once, three operations per dividend".  q[i] must equal the correctly rounded
 * a[i] / b[i] bit for bit for ANY operands (zeros, subnormals, infinities, NaN -> NaN).  a, b, q: n device doubles;
 * needs sstep_cg_create only. */
int sstep_cg_test_division(sstep_cg_t *handle, int64_t n, const double *a, const double *b, double *q);
/* a4, in place: P, AP (interleaved), x, r updated; R_cm(:,1) <- D^-1 r_new; rho_out[0] = ||r_new||^2. */
int sstep_cg_test_update(sstep_cg_t *handle, double *R_cm, const double *AR_cm, double *P_il, double *AP_il,
                         double *x, double *r, const double *beta, const double *alpha, double *rho_out);

/* ---- allocation-free entry point ----
 * Step a2 (M = R^T AR, C = AP^T R, m = R^T r; Eq. 3-4; generalises Alg. 5) for callers that cannot
 * call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.  Needs only
 * sstep_cg_create (no setup, no matrix).  Runs the production gram_kernel on a scratch array that is a STATIC part of
 * the library image (364 544 bytes of every GPU that loads the library, until the process exits): the call itself
 * performs no cudaMalloc / cudaFree and calls no allocating library routine -- three kernel launches on the handle's
 * stream, nothing else; it returns without synchronising.
 *   n >= 1 rows; 1 <= s <= 8 (LIMIT: the static scratch holds 2s^2+s <= 136 entries for at most 320 blocks; larger s is
 *   rejected with SSTEP_CG_ERR_ARG and a text in sstep_cg_last_error).
 *   R_cm, AR_cm: n x s column-major; AP_il: n x s interleaved; r: n   (device, read only)
 *   M, C: s*s row-major; m: s                                          (device, caller-owned outputs)
 * All calls on a device share the one array, which keeps the previous call's contents (the call clears what must start
 * clean); calls that OVERLAP on the GPU -- two streams, two handles on the same device -- race on it: serialise them.
 * Same summation scheme as the solver's Gram kernel (fixed order, reproducible run to run); the grid is capped at 320
 * blocks, so the bits may differ from sstep_cg_test_gram's within the Gram tolerance. */
int sstep_cg_gram_noalloc(sstep_cg_t *handle, int64_t n, int s, const double *R_cm, const double *AR_cm,
                          const double *AP_il, const double *r, double *M, double *C, double *m);

#ifdef __cplusplus
}
#endif
#endif /* SSTEP_CG_H */

// moment.cuh -- the paper-literal scalar work of the s-step PCG (option "form" = 1):
// Alg. 5 (`cvm`) reduced to nothing -- the 2s moments
//     mu^0 = R_1^T r,   mu^{2j-1} = R_j^T AR_j,   mu^{2j} = R_{j+1}^T AR_j        (Eq. 4)
// are accumulated in the epilogues of the matrix-powers SpMVs (mu^0 in the update kernel), so the Gram pass over
// R, AR, AP, r disappears -- and Alg. 6 (`SW`, readings A1-A3 of DESIGN.md) in ONE warp:
//     k = 0 : W = M (Hankel, M(i,j) = mu^{i+j-1}), beta = 0, alpha = W^-1 vm(1:s)
//     k > 0 : rhs by the triangular recurrence from vm and the previous alpha, b1(i,j) = -rhs(i+j-1),
//             beta = W_prev^-1 b1, W = M - b1 beta, alpha = W^-1 vm(1:s)
// Monomial basis only (the Hankel structure assumes it).  Every operation is an explicitly rounded __dmul_rn /
// __dadd_rn / __ddiv_rn in the order Alg. 6 is printed (no FMA contraction), so the result is reproducible bit for bit.
#pragma once
#include "common.cuh"
#include "small_solve.cuh"

struct SwSmem {
    double rhs[2 * SCG_SMAX];
    double b1[SCG_SMAX * SCG_SMAX];
    double bt[SCG_SMAX * SCG_SMAX];
    SmallSolveSmem ss;
};

// Whole warp.  vm: 2s moments (vm[k] = mu^k).  first: k = 0.  alpha/W: in = previous iteration's, out = new.
// Returns 0 or 2 (breakdown).
__device__ inline int warp_sw(int s, bool first, const double* vm, double* beta, double* alpha, double* W, SwSmem& sm,
                              int lane) {
    if (first) {
        for (int e = lane; e < s * s; e += 32) {
            sm.ss.Wn[e] = vm[e / s + e % s + 1];
            beta[e] = 0.0;
        }
        __syncwarp();
    } else {
        const double as = alpha[s - 1];
        if (as == 0.0 || !isfinite(as)) return 2;
        if (lane == 0) {  // Alg. 6 l.1-8: O(s^2) sequential flops
            for (int i = 0; i < 2 * s - 1; i++) sm.rhs[i] = 0.0;
            for (int i = 1; i <= s; i++) {
                double t = vm[i - 1];
                for (int j = 1; j <= i - 1; j++) t = __dadd_rn(t, __dmul_rn(sm.rhs[s - 1 + j - 1], alpha[s - i + j - 1]));
                sm.rhs[s - 1 + i - 1] = __ddiv_rn(-t, as);
            }
        }
        __syncwarp();
        for (int e = lane; e < s * s; e += 32) sm.b1[e] = -sm.rhs[e / s + e % s];  // l.9-13: b1(i,j) = -rhs(i+j-1), full Hankel (A1)
        __syncwarp();
        if (!warp_cholesky(s, W, sm.ss.L, lane)) return 2;
        warp_chol_solve(s, sm.ss.L, s, sm.b1, /*neg=*/false, sm.bt, sm.ss.Y, lane);       // l.14: W_prev beta = b1
        for (int e = lane; e < s * s; e += 32) {                                         // l.15-20: W = M - b1 beta
            const int i = e / s, j = e % s;
            double v = vm[i + j + 1];
            for (int l = 0; l < s; l++) v = __dadd_rn(v, -__dmul_rn(sm.b1[i * s + l], sm.bt[l * s + j]));
            sm.ss.Wn[e] = v;
        }
        __syncwarp();
        for (int e = lane; e < s * s; e += 32) beta[e] = sm.bt[e];
    }
    if (!warp_cholesky(s, sm.ss.Wn, sm.ss.L, lane)) return 2;
    warp_chol_solve(s, sm.ss.L, 1, vm, /*neg=*/false, alpha, sm.ss.Y, lane);             // l.21: W alpha = vm(1:s)
    bool fin = true;
    for (int i = 0; i < s; i++) fin = fin && isfinite(alpha[i]);
    for (int e = lane; e < s * s; e += 32) W[e] = sm.ss.Wn[e];
    __syncwarp();
    return fin ? 0 : 2;
}

// One block after the matrix-powers kernel: sums the per-block moment partials in a fixed order, then the scalar
// work.  mom: [2s][nblk] (row m = partials of mu^m, rows 1..2s-1 used); mu^0 comes from the update / init kernel.
__global__ void __launch_bounds__(256) sw_kernel(int s, int nblk, const double* __restrict__ mom, ScgState* __restrict__ st,
                                                 int do_solve) {
    pdl_wait();  // (common.cuh: the predecessor in the graph may still be draining)
    pdl_launch();
    if (st->status != SCG_RUNNING) return;
    __shared__ double vm[2 * SCG_SMAX];
    __shared__ SwSmem sm;
    __shared__ double al[SCG_SMAX], sW[SCG_SMAX * SCG_SMAX], sbeta[SCG_SMAX * SCG_SMAX];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    // rows 1 .. 2s-1 of mom, two warps-worth of work per moment would not help: one warp per moment, loads overlapped
    for (int m = 1 + warp; m < 2 * s; m += nw) {
        const double v = warp_sum_array(mom + (int64_t)m * nblk, nblk, lane);
        if (lane == 0) vm[m] = v;
    }
    if (threadIdx.x == 0) vm[0] = st->mu0;
    if (threadIdx.x < s) al[threadIdx.x] = st->alpha[threadIdx.x];
    for (int e = threadIdx.x; e < s * s; e += blockDim.x) sW[e] = st->W[e];
    __syncthreads();
    if (warp == 0) {
        for (int e = lane; e < 2 * s; e += 32) st->vm[e] = vm[e];
        if (do_solve) {  // all operands in shared memory: Alg. 6 is one long dependent chain
            const int rc = warp_sw(s, st->k == 0, vm, sbeta, al, sW, sm, lane);
            for (int e = lane; e < s * s; e += 32) { st->W[e] = sW[e]; st->beta[e] = sbeta[e]; }
            if (lane < s) st->alpha[lane] = al[lane];
            if (lane == 0 && rc != 0) st->status = rc;
        }
    }
}

// stand-alone Alg. 6 for the test hook: operands in global memory
__global__ void sw_test_kernel(int s, int first, const double* vm, double* beta, double* alpha, double* W, int* status_out) {
    __shared__ SwSmem sm;
    const int rc = warp_sw(s, first != 0, vm, beta, alpha, W, sm, threadIdx.x);
    if (threadIdx.x == 0) status_out[0] = rc;
}

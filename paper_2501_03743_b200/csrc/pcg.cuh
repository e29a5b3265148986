// pcg.cuh -- SURVEY.md 8(f) NEXT-3: the textbook preconditioned CG of Alg. 1 (PCG-HS) as its own kernel
// sequence (option "method" = 1), the classical comparator with TWO reductions per iteration:
//   K1  s_k = A p_k, with the per-block partials of p_k^T s_k in the SpMV epilogue        (spmv.cuh, moment epilogue)
//   K2  alpha_k = u_k^T r_k / p_k^T s_k ; x += alpha p ; r -= alpha s ; u = D^-1 r ; partials of u^T r and r^T r ;
//       cross-block finish: beta_k = u_{k+1}^T r_{k+1} / u_k^T r_k, k <- k + 1, stop test ||r|| < rtol ||r_0||
//   K3  p = u + beta_k p
// Workspaces of the s-step path at s = 1 are reused: p = P, s = AP, u = R(:,1); u^T r lives in ScgState::mu0,
// alpha / beta in ScgState::alpha[0] / beta[0].  HBM bytes per iteration: CSR + 8n (2 + 7 + 3).
#pragma once
#include "common.cuh"
#include "update.cuh"

// K2.  ps_partials: [nps] per-block partials of p^T s left by the SpMV (summed here by EVERY block in the same fixed
// order, so all blocks use the same alpha).  partials: [2][gridDim.x] scratch for u^T r and r^T r.
__global__ void __launch_bounds__(256, 4)
pcg_update_kernel(int64_t n, const double* __restrict__ p, const double* __restrict__ sk, double* __restrict__ x,
                  double* __restrict__ r, double* __restrict__ u, const double* __restrict__ dinv,
                  const double* __restrict__ ps_partials, int nps, double* __restrict__ partials, ScgState* __restrict__ st,
                  double dinv_uniform) {
    if (st->status != SCG_RUNNING) return;
    __shared__ double s_alpha;
    __shared__ double red[2][8];
    __shared__ bool is_last;
    if (threadIdx.x < 32) {
        const double ps = warp_sum_array(ps_partials, nps, (int)threadIdx.x);
        if (threadIdx.x == 0) s_alpha = (ps > 0.0 && isfinite(ps)) ? st->mu0 / ps : nan("");
    }
    __syncthreads();
    const double alpha = s_alpha;
    if (!isfinite(alpha)) {  // p^T A p <= 0 or not finite: breakdown, x keeps the last iterate (every block decides alike)
        if (blockIdx.x == 0 && threadIdx.x == 0) st->status = 2;
        return;
    }
    double ur = 0.0, rr = 0.0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    // two rows per thread as 128-bit vectors (all operands are cudaMalloc'ed workspaces: 16-byte aligned); odd tail below
    const int64_t n2 = n >> 1;
    const double2* p2 = reinterpret_cast<const double2*>(p);
    const double2* s2 = reinterpret_cast<const double2*>(sk);
    const double2* d2 = reinterpret_cast<const double2*>(dinv);
    double2* x2 = reinterpret_cast<double2*>(x);
    double2* r2 = reinterpret_cast<double2*>(r);
    double2* u2 = reinterpret_cast<double2*>(u);
    auto one = [&](double2 pi, double2 si, double2 di, double2 xi, double2 ri, int64_t i) {
        double2 ui;
        xi.x = fma(alpha, pi.x, xi.x); xi.y = fma(alpha, pi.y, xi.y);
        ri.x = fma(-alpha, si.x, ri.x); ri.y = fma(-alpha, si.y, ri.y);
        ui.x = di.x * ri.x; ui.y = di.y * ri.y;
        x2[i] = xi; r2[i] = ri; u2[i] = ui;
        ur = fma(ui.x, ri.x, ur); ur = fma(ui.y, ri.y, ur);
        rr = fma(ri.x, ri.x, rr); rr = fma(ri.y, ri.y, rr);
    };
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + stride < n2; i += 2 * stride) {  // two independent row pairs per trip: ten 128-bit loads in flight
        const int64_t j = i + stride;
        const double2 pa = ldg_stream2(reinterpret_cast<const double*>(p2 + i)), pb = ldg_stream2(reinterpret_cast<const double*>(p2 + j));
        const double2 sa = ldg_stream2(reinterpret_cast<const double*>(s2 + i)), sb = ldg_stream2(reinterpret_cast<const double*>(s2 + j));
        const double2 da = (dinv_uniform > 0.0) ? make_double2(dinv_uniform, dinv_uniform) : d2[i];
        const double2 db = (dinv_uniform > 0.0) ? da : d2[j];
        const double2 xa = x2[i], xb = x2[j];
        const double2 ra = r2[i], rb = r2[j];
        one(pa, sa, da, xa, ra, i);
        one(pb, sb, db, xb, rb, j);
    }
    if (i < n2)
        one(ldg_stream2(reinterpret_cast<const double*>(p2 + i)), ldg_stream2(reinterpret_cast<const double*>(s2 + i)),
            (dinv_uniform > 0.0) ? make_double2(dinv_uniform, dinv_uniform) : d2[i], x2[i], r2[i], i);
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const int64_t row = n - 1;
        const double xi = fma(alpha, p[row], x[row]);
        const double ri = fma(-alpha, sk[row], r[row]);
        const double ui = dinv[row] * ri;
        x[row] = xi; r[row] = ri; u[row] = ui;
        ur = fma(ui, ri, ur);
        rr = fma(ri, ri, rr);
    }
    ur = warp_sum(ur);
    rr = warp_sum(rr);
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = ur; red[1][threadIdx.x >> 5] = rr; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) { a += red[0][w]; b += red[1][w]; }
        partials[blockIdx.x] = a;
        partials[gridDim.x + blockIdx.x] = b;
        __threadfence();
        const unsigned int t = atomicAdd(&st->ticket_update, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    if (threadIdx.x < 32) {
        __threadfence();
        const double a = warp_sum_array(partials, (int)gridDim.x, (int)threadIdx.x);
        const double b = warp_sum_array(partials + gridDim.x, (int)gridDim.x, (int)threadIdx.x);
        if (threadIdx.x == 0) {
            st->alpha[0] = alpha;
            st->beta[0] = a / st->mu0;  // beta_k = u_{k+1}^T r_{k+1} / u_k^T r_k
            st->mu0 = a;
            st->rho = b;
            st->k = st->k + 1;
            if (!isfinite(b) || !isfinite(a)) st->status = 2;
            else if (sqrt(b) < st->rtol * sqrt(st->rho0)) st->status = 0;
            st->ticket_update = 0;
        }
    }
}

// K3: p = u + beta p
__global__ void __launch_bounds__(256, 4)
pcg_direction_kernel(int64_t n, const double* __restrict__ u, double* __restrict__ p, const ScgState* __restrict__ st) {
    if (st->status != SCG_RUNNING) return;
    const double beta = st->beta[0];
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t n2 = n >> 1;
    double2* p2 = reinterpret_cast<double2*>(p);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += stride) {
        const double2 ui = ldg_stream2(u + 2 * i);
        double2 pi = p2[i];
        pi.x = fma(beta, pi.x, ui.x);
        pi.y = fma(beta, pi.y, ui.y);
        p2[i] = pi;
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) p[n - 1] = fma(beta, p[n - 1], u[n - 1]);
}

// update.cuh -- step a4 (+ the stop test a5): the fused tall-skinny block updates of Alg. 3 l.17-21
// (PAPER.md:158), every n x s block streamed exactly once (the paper's "Dgemmv" idea):
//   P  <- R  + P  beta        x <- x + P  alpha
//   AP <- AR + AP beta        r <- r - AP alpha
// plus, fused by this build so no extra pass is needed: R(:,1) <- D^-1 r (the next MPK's first column),
// rho = ||r||^2 with a deterministic single-kernel cross-block finish, k <- k+1 and the stop test
// ||r|| < rtol ||r_0|| (Alg. 3 l.31-33).
// Layout: R, AR column-major; P, AP interleaved (one row = s consecutive doubles = 128-bit loads/stores).
// One thread per row; beta (s x s) and alpha (s) are broadcast from shared memory.
#pragma once
#include "common.cuh"

// V_new(row, :) = Xcol(row, :) + V(row, :) beta ; acc += sign * V_new(row, :) alpha.  Per output column the sum runs
// over l in ascending order and acc over j in ascending order (the order of update_half); beta is read from shared
// memory as 128-bit pairs (two output columns per load).
template <int S>
__device__ __forceinline__ double update_row(const double (&v)[S], double (&out)[S], const double* sbeta,
                                             const double* salpha, double acc, double sign) {
    if constexpr (S % 2 == 0) {
#pragma unroll
        for (int l = 0; l < S; l++) {
            const double2* b2 = reinterpret_cast<const double2*>(sbeta + l * S);
#pragma unroll
            for (int j = 0; j < S / 2; j++) {
                const double2 b = b2[j];
                out[2 * j] = fma(v[l], b.x, out[2 * j]);
                out[2 * j + 1] = fma(v[l], b.y, out[2 * j + 1]);
            }
        }
    } else {
#pragma unroll
        for (int l = 0; l < S; l++)
#pragma unroll
            for (int j = 0; j < S; j++) out[j] = fma(v[l], sbeta[l * S + j], out[j]);
    }
#pragma unroll
    for (int j = 0; j < S; j++) acc = fma(sign * out[j], salpha[j], acc);
    return acc;
}

template <int S>
__device__ __forceinline__ void store_row(double* __restrict__ dst, const double (&out)[S]) {
    if constexpr (S % 2 == 0) {
        double2* d2 = reinterpret_cast<double2*>(dst);
#pragma unroll
        for (int l = 0; l < S / 2; l++) d2[l] = make_double2(out[2 * l], out[2 * l + 1]);
    } else {
#pragma unroll
        for (int l = 0; l < S; l++) dst[l] = out[l];
    }
}

// one half of the update for one row: V <- Xcol + V beta (V = P or AP, interleaved), acc <- acc + sign * (V_new alpha)
template <int S>
__device__ __forceinline__ double update_half(int64_t n, int64_t row, const double* __restrict__ Xcm, double* __restrict__ Vil,
                                              const volatile double* sbeta, const double* salpha, double acc, double sign) {
    // sbeta is read through a volatile pointer on purpose: it stops the compiler from hoisting all S*S entries into
    // registers across the row loop (which costs the occupancy this bandwidth-bound kernel lives on)
    double v[S], out[S];
    if constexpr (S % 2 == 0) {
        const double2* v2 = reinterpret_cast<const double2*>(Vil + row * S);
#pragma unroll
        for (int l = 0; l < S / 2; l++) {
            const double2 a = v2[l];
            v[2 * l] = a.x;
            v[2 * l + 1] = a.y;
        }
    } else {
#pragma unroll
        for (int l = 0; l < S; l++) v[l] = Vil[row * S + l];
    }
#pragma unroll
    for (int j = 0; j < S; j++) out[j] = Xcm[(int64_t)j * n + row];
#pragma unroll
    for (int j = 0; j < S; j++) {
        double p = out[j];
#pragma unroll
        for (int l = 0; l < S; l++) p = fma(v[l], sbeta[l * S + j], p);
        out[j] = p;
        acc = fma(sign * p, salpha[j], acc);
    }
    if constexpr (S % 2 == 0) {
        double2* v2 = reinterpret_cast<double2*>(Vil + row * S);
#pragma unroll
        for (int l = 0; l < S / 2; l++) v2[l] = make_double2(out[2 * l], out[2 * l + 1]);
    } else {
#pragma unroll
        for (int l = 0; l < S; l++) Vil[row * S + l] = out[l];
    }
    return acc;
}

// ---- ||r||^2 (and mu^0 = R_1^T r of the moment form) finish shared by the update kernels: block reduce over the first
// `nw` warps, per-block partials, ticket, fixed-order sum in the last block, then k <- k + 1 and the stop test
// (Alg. 3 l.31-33).  partials: [2][gridDim.x].  Every thread of the CTA calls.  MOM: only the moment form pays for mu^0.
template <bool MOM>
__device__ __forceinline__ void update_block_finish(double rho, double mu0, int nw, double* __restrict__ partials,
                                                    ScgState* __restrict__ st, double* __restrict__ rho_out,
                                                    bool count_iteration = true) {
    __shared__ double red[MOM ? 2 : 1][32];
    __shared__ bool is_last;
    rho = warp_sum(rho);
    if (MOM) mu0 = warp_sum(mu0);
    if ((threadIdx.x & 31) == 0 && (int)(threadIdx.x >> 5) < nw) {
        red[0][threadIdx.x >> 5] = rho;
        if (MOM) red[MOM ? 1 : 0][threadIdx.x >> 5] = mu0;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0.0, w = 0.0;
        for (int i = 0; i < nw; i++) { v += red[0][i]; if (MOM) w += red[MOM ? 1 : 0][i]; }
        partials[blockIdx.x] = v;
        if (MOM) partials[gridDim.x + blockIdx.x] = w;
        __threadfence();
        const unsigned int t = atomicAdd(&st->ticket_update, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    if (threadIdx.x < 32) {
        __threadfence();
        const double v = warp_sum_array(partials, (int)gridDim.x, (int)threadIdx.x);
        double w = 0.0;
        if (MOM) w = warp_sum_array(partials + gridDim.x, (int)gridDim.x, (int)threadIdx.x);
        if (threadIdx.x == 0) {
            st->rho = v;
            if (MOM) st->mu0 = w;
            if (count_iteration) st->k = st->k + 1;
            if (rho_out) rho_out[0] = v;
            if (!isfinite(v)) st->status = 2;
            else if (sqrt(v) < st->rtol * sqrt(st->rho0)) st->status = 0;
            st->ticket_update = 0;
        }
    }
}

template <int S, bool MOM>
// Occupancy: three CTAs per SM for s = 3, 4 (80 registers, no spills): 768 rows x 144 bytes of loads in flight per SM
// instead of 512 -- update<4> on 320^3 1221 -> 1165 us (6.5 TB/s, the copy peak); larger s (hooks on misaligned buffers
// only -- the staged kernel serves s >= 5) keep two.
__global__ void __launch_bounds__(256, (S <= 2) ? 4 : (S <= 4) ? 3 : 2)
update_kernel(int64_t n, double* __restrict__ R, const double* __restrict__ AR, double* __restrict__ P,
              double* __restrict__ AP, double* __restrict__ x, double* __restrict__ r, const double* __restrict__ dinv,
              const double* __restrict__ beta_g, const double* __restrict__ alpha_g, double* __restrict__ partials,
              ScgState* __restrict__ st, double* __restrict__ rho_out, double dinv_uniform) {
    pdl_wait();  // (common.cuh: the predecessor in the graph may still be draining)
    pdl_launch();
    if (st->status != SCG_RUNNING) return;
    __shared__ __align__(16) double sbeta[S * S];
    __shared__ double salpha[S];
    for (int e = threadIdx.x; e < S * S; e += blockDim.x) sbeta[e] = beta_g[e];
    if (threadIdx.x < S) salpha[threadIdx.x] = alpha_g[threadIdx.x];
    __syncthreads();

    double rho = 0.0, mu0 = 0.0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; row < n; row += stride) {
        // (a constant diagonal -- every Poisson config -- needs no dinv stream: 8n bytes less per update)
        const double x0 = x[row], r0 = r[row], di = (dinv_uniform > 0.0) ? dinv_uniform : dinv[row];
        const double xi = update_half<S>(n, row, R, P, sbeta, salpha, x0, 1.0);     // P <- R + P beta ; x += P alpha
        const double ri = update_half<S>(n, row, AR, AP, sbeta, salpha, r0, -1.0);  // AP <- AR + AP beta ; r -= AP alpha
        x[row] = xi;
        r[row] = ri;
        const double r1 = di * ri;
        R[row] = r1;  // R(:,1) of the next outer iteration
        rho = fma(ri, ri, rho);
        if (MOM) mu0 = fma(r1, ri, mu0);  // moment form: mu^0 = R_1^T r
    }
    update_block_finish<MOM>(rho, mu0, (int)(blockDim.x >> 5), partials, st, rho_out);
}

// ---- s = 1: every stream (R, AR, P, AP, x, r) is a plain contiguous vector, and six 8-byte loads per thread leave too few
// bytes in flight (update_kernel<1> ran at 0.89 of the copy peak on 320^3).  Two consecutive rows per thread, 128-bit
// loads and stores: twice the bytes in flight at the same occupancy.  Per row the same operations in the same order as
// update_half<1>; needs 16-byte aligned buffers (the caller falls back to update_kernel<1> otherwise).
template <bool MOM>
__global__ void __launch_bounds__(256, 4)
update1_kernel(int64_t n, double* __restrict__ R, const double* __restrict__ AR, double* __restrict__ P,
               double* __restrict__ AP, double* __restrict__ x, double* __restrict__ r, const double* __restrict__ dinv,
               const double* __restrict__ beta_g, const double* __restrict__ alpha_g, double* __restrict__ partials,
               ScgState* __restrict__ st, double* __restrict__ rho_out, double dinv_uniform) {
    pdl_wait();
    pdl_launch();
    if (st->status != SCG_RUNNING) return;
    const double beta = beta_g[0], alpha = alpha_g[0];
    double rho = 0.0, mu0 = 0.0;
    const int64_t npairs = n >> 1;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    auto one_row = [&](double Rv, double ARv, double Pv, double APv, double xv, double rv, double di, double& Pn, double& APn,
                       double& xn, double& rn, double& r1) {
        Pn = fma(Pv, beta, Rv);          // P <- R + P beta
        xn = fma(Pn, alpha, xv);         // x += P alpha        (update_half: acc = fma(sign * p, alpha, acc), sign = +1)
        APn = fma(APv, beta, ARv);       // AP <- AR + AP beta
        rn = fma(-1.0 * APn, alpha, rv); // r -= AP alpha       (sign = -1)
        r1 = di * rn;
        rho = fma(rn, rn, rho);
        if (MOM) mu0 = fma(r1, rn, mu0);
    };
    for (int64_t pr = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; pr < npairs; pr += stride) {
        const int64_t row = 2 * pr;
        const double2 Rv = *reinterpret_cast<const double2*>(R + row), ARv = *reinterpret_cast<const double2*>(AR + row);
        const double2 Pv = *reinterpret_cast<const double2*>(P + row), APv = *reinterpret_cast<const double2*>(AP + row);
        const double2 xv = *reinterpret_cast<const double2*>(x + row), rv = *reinterpret_cast<const double2*>(r + row);
        double2 di = make_double2(dinv_uniform, dinv_uniform);
        if (!(dinv_uniform > 0.0)) di = *reinterpret_cast<const double2*>(dinv + row);
        double2 Pn, APn, xn, rn, r1;
        one_row(Rv.x, ARv.x, Pv.x, APv.x, xv.x, rv.x, di.x, Pn.x, APn.x, xn.x, rn.x, r1.x);
        one_row(Rv.y, ARv.y, Pv.y, APv.y, xv.y, rv.y, di.y, Pn.y, APn.y, xn.y, rn.y, r1.y);
        *reinterpret_cast<double2*>(P + row) = Pn;
        *reinterpret_cast<double2*>(AP + row) = APn;
        *reinterpret_cast<double2*>(x + row) = xn;
        *reinterpret_cast<double2*>(r + row) = rn;
        *reinterpret_cast<double2*>(R + row) = r1;  // R(:,1) of the next outer iteration
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {  // odd n: the last row
        const int64_t row = n - 1;
        const double di = (dinv_uniform > 0.0) ? dinv_uniform : dinv[row];
        double Pn, APn, xn, rn, r1;
        one_row(R[row], AR[row], P[row], AP[row], x[row], r[row], di, Pn, APn, xn, rn, r1);
        P[row] = Pn; AP[row] = APn; x[row] = xn; r[row] = rn; R[row] = r1;
    }
    update_block_finish<MOM>(rho, mu0, (int)(blockDim.x >> 5), partials, st, rho_out);
}

// ---- residual replacement (option "replace_every", reading A22): r <- b - A x with y = A x from the
// production SpMV, R(:,1) <- D^-1 r, rho = ||r||^2 and the stop test taken again on the replaced residual.  P, AP stay.
__global__ void __launch_bounds__(256)
replace_kernel(int64_t n, const double* __restrict__ b, const double* __restrict__ y, double* __restrict__ r,
               double* __restrict__ R1, const double* __restrict__ dinv, double* __restrict__ partials,
               ScgState* __restrict__ st) {
    if (st->status != SCG_RUNNING) return;
    double rho = 0.0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; row < n; row += stride) {
        const double ri = b[row] - y[row];
        r[row] = ri;
        R1[row] = dinv[row] * ri;
        rho = fma(ri, ri, rho);
    }
    update_block_finish<false>(rho, 0.0, (int)(blockDim.x >> 5), partials, st, nullptr, /*count_iteration=*/false);
}

// ---- start of a solve: r = b - A x0 (Ax0 already in r if have_ax), x = x0, R(:,1) = D^-1 r, rho0 = ||r||^2 ----
__global__ void __launch_bounds__(256)
init_kernel(int64_t n, const double* __restrict__ b, const double* __restrict__ x0, int have_ax, double* __restrict__ x,
            double* __restrict__ r, double* __restrict__ R, const double* __restrict__ dinv, double* __restrict__ partials,
            ScgState* __restrict__ st, int s, double rtol) {
    __shared__ double red[2][8];
    __shared__ bool is_last;
    double rho = 0.0, mu0 = 0.0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; row < n; row += stride) {
        const double ri = have_ax ? b[row] - r[row] : b[row];
        const double r1 = dinv[row] * ri;
        x[row] = x0 ? x0[row] : 0.0;
        r[row] = ri;
        R[row] = r1;
        rho = fma(ri, ri, rho);
        mu0 = fma(r1, ri, mu0);
    }
    rho = warp_sum(rho);
    mu0 = warp_sum(mu0);
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = rho; red[1][threadIdx.x >> 5] = mu0; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0.0, u = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) { v += red[0][w]; u += red[1][w]; }
        partials[blockIdx.x] = v;
        partials[gridDim.x + blockIdx.x] = u;
        __threadfence();
        const unsigned int t = atomicAdd(&st->ticket_init, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    if (threadIdx.x < 32) {
        __threadfence();
        const double v = warp_sum_array(partials, (int)gridDim.x, (int)threadIdx.x);
        const double u = warp_sum_array(partials + gridDim.x, (int)gridDim.x, (int)threadIdx.x);
        for (int e = threadIdx.x; e < s * s; e += 32) {
            st->W[e] = (e / s == e % s) ? 1.0 : 0.0;  // W_prev = I with C = 0 gives beta = 0, W = M at k = 0
            st->Lw[e] = (e / s == e % s) ? 1.0 : 0.0;  // its Cholesky factor (sqrt(1) = 1: the bits warp_cholesky gives)
            st->beta[e] = 0.0;
        }
        if (threadIdx.x == 0) {
            st->rho = v;
            st->rho0 = v;
            st->mu0 = u;
            st->rtol = rtol;
            st->k = 0;
            st->status = (v == 0.0) ? 0 : (isfinite(v) ? SCG_RUNNING : 2);
            st->ticket_init = 0;
            st->ticket_gram = 0;
            st->ticket_update = 0;
        }
    }
}

// ---- setup: is the diagonal constant?  flag[0] stays 1 if every dinv[i] has the bits of dinv[0]
__global__ void uniform_diag_kernel(int64_t n, const double* __restrict__ dinv, int* __restrict__ flag) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool bad = (i < n) && (dinv[i] != dinv[0]);
    if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicAnd(flag, 0);
}

// ---- setup: dinv = 1/a_ii, structural validation, row-length statistics ----
// err bits: 1 = rowptr not monotone / out of range, 2 = column index out of range, 4 = diagonal missing, duplicated or <= 0
__global__ void analyze_kernel(int64_t n, int64_t nnz, const int* __restrict__ rp, const int* __restrict__ ci,
                               const double* __restrict__ va, double* __restrict__ dinv, int* __restrict__ err,
                               int* __restrict__ max_len) {
    const int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int e = 0, len = 0;
    if (row < n) {
        const int lo = rp[row], hi = rp[row + 1];
        if (lo < 0 || hi < lo || hi > nnz || (row == 0 && lo != 0) || (row == n - 1 && hi != nnz)) e |= 1;
        double d = 0.0;
        int found = 0;  // the diagonal entry must appear exactly once (the bulk SpMV takes 1/a_ii from the row itself)
        if (!e) {
            len = hi - lo;
            for (int k = lo; k < hi; k++) {
                const int c = ci[k];
                if (c < 0 || c >= n) e |= 2;
                if (c == row) { d = va[k]; found++; }
            }
            if (found != 1 || !(d > 0.0)) e |= 4;
        }
        dinv[row] = (e == 0) ? 1.0 / d : 0.0;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        e |= __shfl_xor_sync(0xffffffffu, e, o);
        len = max(len, __shfl_xor_sync(0xffffffffu, len, o));
    }
    if ((threadIdx.x & 31) == 0) {
        if (e) atomicOr(err, e);
        atomicMax(max_len, len);
    }
}

// Interleave / de-interleave helpers for the Python binding's marshalling are NOT provided: the binding
// transposes with torch; the kernels only ever see the documented layouts.

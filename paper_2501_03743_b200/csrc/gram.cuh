// gram.cuh -- steps a2 + a3: the fused block inner products of one outer iteration in ONE pass over HBM,
//   M = R^T AR (s x s),  C = AP^T R (s x s),  m = R^T r (s)      (Eq. 3-4; generalises Alg. 5)
// followed, in the same kernel, by a deterministic cross-block finish and the s x s solves in one warp of the
// last block to arrive (replaces the paper's device->host copy + MPI_Allreduce + CPU solve).
//
// Layout: R, AR column-major (column j at X + j*n); AP interleaved (row i at AP + i*s).
// Work split: a thread owns one row at a time and a SLICE of G consecutive columns q*G..q*G+G-1 of AR / AP:
//   accM[i][g] += R_i * AR_{qG+g}   (S x G)      accC[g][j] += AP_{qG+g} * R_j   (G x S)      accm[g] += R_{qG+g} * r
// so 2*S*G + G accumulators stay in registers (<= 39 doubles for every S <= 16).  The NSL = ceil(S/G) slices of
// one row group are warps of the same CTA reading the same R rows at the same time (L1 hits).
#pragma once
#include "common.cuh"
#include "small_solve.cuh"

template <int S>
struct GramCfg {
    static constexpr int G = (S <= 4) ? S : (S <= 6) ? 3 : (S <= 9) ? 2 : 1;
    static constexpr int NSL = (S + G - 1) / G;             // slices
    static constexpr int RG = (NSL >= 8) ? 1 : 8 / NSL;     // row groups (warps per slice) per CTA
    static constexpr int NW = NSL * RG;                     // warps per CTA
    static constexpr int NACC = 2 * S * G + G;              // accumulators per thread
    static constexpr int NE = 2 * S * S + S;                // Gram entries: M | C | m
};

// entry index of accumulator a of slice q
template <int S>
__device__ __forceinline__ int gram_entry(int q, int a, bool& valid) {
    constexpr int G = GramCfg<S>::G;
    if (a < S * G) {  // accM[i][g]
        const int i = a / G, col = q * G + a % G;
        valid = col < S;
        return i * S + col;
    } else if (a < 2 * S * G) {  // accC[g][j]
        const int b = a - S * G;
        const int row = q * G + b / S, j = b % S;
        valid = row < S;
        return S * S + row * S + j;
    }
    const int col = q * G + (a - 2 * S * G);
    valid = col < S;
    return 2 * S * S + col;
}

template <int S>
__global__ void __launch_bounds__(GramCfg<S>::NW * 32)
gram_kernel(int64_t n, const double* __restrict__ R, const double* __restrict__ AR, const double* __restrict__ AP,
            const double* __restrict__ r, double* __restrict__ partials, ScgState* __restrict__ st, int do_solve, int pf) {
    using Cfg = GramCfg<S>;
    constexpr int G = Cfg::G, NSL = Cfg::NSL, RG = Cfg::RG, NW = Cfg::NW, NACC = Cfg::NACC, NE = Cfg::NE;
    if (st->status != SCG_RUNNING) return;
    __shared__ double red[NW][NACC];
    __shared__ double fin[NE];
    __shared__ SmallSolveSmem ssm;
    __shared__ bool is_last;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int q = warp % NSL;   // slice
    const int rg = warp / NSL;  // row group
    double accM[S][G], accC[G][S], accm[G];
#pragma unroll
    for (int g = 0; g < G; g++) {
        accm[g] = 0.0;
#pragma unroll
        for (int i = 0; i < S; i++) { accM[i][g] = 0.0; accC[g][i] = 0.0; }
    }
    const int c0 = q * G;
    const int64_t stride = (int64_t)gridDim.x * RG * 32;
    for (int64_t row = ((int64_t)blockIdx.x * RG + rg) * 32 + lane; row < n; row += stride) {
        double Rv[S], ARv[G], APv[G], Rsel[G];
        if (pf > 0) {  // pull the rows this thread reads `pf` iterations from now into L2 (hides the DRAM latency)
            const int64_t prow = row + pf * stride;
            if (prow < n) {
                if (q == 0) {
#pragma unroll
                    for (int j = 0; j < S; j++) prefetch_l2(R + (int64_t)j * n + prow);
                    prefetch_l2(r + prow);
                }
#pragma unroll
                for (int g = 0; g < G; g++)
                    if ((G * NSL == S) || (c0 + g < S)) prefetch_l2(AR + (int64_t)(c0 + g) * n + prow);
                prefetch_l2(AP + prow * S + c0);
            }
        }
#pragma unroll
        for (int j = 0; j < S; j++) Rv[j] = R[(int64_t)j * n + row];
#pragma unroll
        for (int g = 0; g < G; g++) {
            const bool ok = (G * NSL == S) || (c0 + g < S);
            ARv[g] = ok ? AR[(int64_t)(c0 + g) * n + row] : 0.0;
            APv[g] = ok ? AP[row * S + c0 + g] : 0.0;
            Rsel[g] = ok ? R[(int64_t)(c0 + g) * n + row] : 0.0;  // R_{c0+g} again (L1 hit): keeps Rv[] statically indexed
        }
        const double rv = r[row];
#pragma unroll
        for (int g = 0; g < G; g++) {
#pragma unroll
            for (int i = 0; i < S; i++) {
                accM[i][g] = fma(Rv[i], ARv[g], accM[i][g]);
                accC[g][i] = fma(APv[g], Rv[i], accC[g][i]);
            }
            accm[g] = fma(Rsel[g], rv, accm[g]);
        }
    }
    // ---- block reduction: shuffle tree inside the warp, then across the RG row groups of a slice ----
#pragma unroll
    for (int g = 0; g < G; g++) {
#pragma unroll
        for (int i = 0; i < S; i++) {
            const double a = warp_sum(accM[i][g]);
            const double b = warp_sum(accC[g][i]);
            if (lane == 0) { red[warp][i * G + g] = a; red[warp][S * G + g * S + i] = b; }
        }
        const double c = warp_sum(accm[g]);
        if (lane == 0) red[warp][2 * S * G + g] = c;
    }
    __syncthreads();
    for (int e = threadIdx.x; e < NSL * NACC; e += blockDim.x) {
        const int qs = e / NACC, a = e % NACC;
        double v = 0.0;
#pragma unroll
        for (int g2 = 0; g2 < RG; g2++) v += red[g2 * NSL + qs][a];
        bool valid;
        const int ge = gram_entry<S>(qs, a, valid);
        if (valid) partials[(int64_t)ge * gridDim.x + blockIdx.x] = v;
    }
    // ---- single-kernel cross-block finish: ticket, last block sums the partials in a fixed order ----
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned int t = atomicAdd(&st->ticket_gram, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    for (int e = warp; e < NE; e += NW) {
        double v = 0.0;
        for (int b = lane; b < (int)gridDim.x; b += 32) v += __ldcg(&partials[(int64_t)e * gridDim.x + b]);
        v = warp_sum(v);
        if (lane == 0) fin[e] = v;
    }
    __syncthreads();
    if (warp == 0) {
        for (int e = lane; e < S * S; e += 32) { st->M[e] = fin[e]; st->C[e] = fin[S * S + e]; }
        if (lane < S) st->m[lane] = fin[2 * S * S + lane];
        if (do_solve) {
            const int rc = warp_small_solve(S, fin, fin + S * S, fin + 2 * S * S, st->W, st->beta, st->alpha, st->W, ssm, lane);
            if (lane == 0 && rc != 0) st->status = rc;
        }
        if (lane == 0) st->ticket_gram = 0;  // re-arm for the next graph replay
    }
}

// stand-alone a3 for the test hook: same device function, operands in global memory
__global__ void small_solve_kernel(int s, const double* M, const double* C, const double* m, const double* Wprev, double* beta,
                                   double* alpha, double* W, int* status_out) {
    __shared__ SmallSolveSmem ssm;
    const int rc = warp_small_solve(s, M, C, m, Wprev, beta, alpha, W, ssm, threadIdx.x);
    if (threadIdx.x == 0) status_out[0] = rc;
}

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

// entry index (in M | C | m) of accumulator a of slice q, for slices of G columns
template <int S, int G>
__device__ __forceinline__ int gram_entry(int q, int a, bool& valid) {
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

// ---- everything after the in-warp reduction.  red[g2 * NSL + q][a] holds, for NRED row groups g2 and NSL slices q,
// the partial sums of the CTA (accumulator order: accM[i][g] at i*G+g, accC[g][i] at S*G+g*S+i, accm[g] at 2*S*G+g).
// Sums the row groups, writes the per-block partials, takes a ticket; the last block sums all partials in a fixed
// order (bitwise reproducible) and one warp runs the s x s solves.  Every thread of the CTA must call (barriers).
template <int S, int G, int NSL, int NRED>
__device__ __forceinline__ void gram_cross_block_finish(const double (*red)[2 * S * G + G], double* __restrict__ partials,
                                                        ScgState* __restrict__ st, int do_solve) {
    constexpr int NACC = 2 * S * G + G, NE = 2 * S * S + S;
    __shared__ double fin[NE];
    __shared__ SmallSolveSmem ssm;
    __shared__ bool is_last;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    __syncthreads();
    for (int e = threadIdx.x; e < NSL * NACC; e += blockDim.x) {
        const int qs = e / NACC, a = e % NACC;
        double v = 0.0;
#pragma unroll
        for (int g2 = 0; g2 < NRED; g2++) v += red[g2 * NSL + qs][a];
        bool valid;
        const int ge = gram_entry<S, G>(qs, a, valid);
        if (valid) partials[(int64_t)ge * gridDim.x + blockIdx.x] = v;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned int t = atomicAdd(&st->ticket_gram, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    __shared__ double sW[S * S], sbeta[S * S], salpha[S];
    // a warp owns the entries warp, warp + nwarps, ...; up to three of them per pass, their loads in flight together
    // (KB = 1, 2 for s = 1, 2: no more registers than the streaming loop of those kernels needs)
    constexpr int KB = (NE <= 8) ? 1 : (NE <= 16) ? 2 : 3;
    // the last warp also fetches the Cholesky factor of the previous outer iteration's W: loads issued before its share of
    // the sums, so that their latency is not added to the chain sums -> barrier -> solves
    constexpr int NLQ = (S * S + 31) / 32;
    double lreg[NLQ];
    if (warp == nwarps - 1) {
#pragma unroll
        for (int q = 0; q < NLQ; q++) lreg[q] = (lane + 32 * q < S * S) ? st->Lw[lane + 32 * q] : 0.0;
    }
    for (int e = warp; e < NE; e += KB * nwarps) {
        double v[KB];
        const int kv = (NE - e + nwarps - 1) / nwarps;
        warp_sum_arrays<KB>(partials + (int64_t)e * gridDim.x, (int64_t)nwarps * gridDim.x, kv < KB ? kv : KB, (int)gridDim.x, lane, v);
        if (lane == 0) {
#pragma unroll
            for (int q = 0; q < KB; q++)
                if (e + q * nwarps < NE) fin[e + q * nwarps] = v[q];
        }
    }
    if (warp == nwarps - 1) {
#pragma unroll
        for (int q = 0; q < NLQ; q++)
            if (lane + 32 * q < S * S) ssm.L[lane + 32 * q] = lreg[q];
    }
    __syncthreads();
    if (warp == 0) {
        for (int e = lane; e < S * S; e += 32) { st->M[e] = fin[e]; st->C[e] = fin[S * S + e]; }
        if (lane < S) st->m[lane] = fin[2 * S * S + lane];
        if (do_solve) {  // all operands in shared memory: the solves are one long dependent chain
            const int rc = warp_small_solve(S, fin, fin + S * S, fin + 2 * S * S, nullptr, sbeta, salpha, sW, ssm, lane, /*have_L=*/true);
            if (rc == 0)
                for (int e = lane; e < S * S; e += 32) st->Lw[e] = ssm.L[e];
            for (int e = lane; e < S * S; e += 32) { st->W[e] = sW[e]; st->beta[e] = sbeta[e]; }
            if (lane < S) st->alpha[lane] = salpha[lane];
            if (lane == 0 && rc != 0) st->status = rc;
        }
        if (lane == 0) st->ticket_gram = 0;  // re-arm for the next graph replay
    }
}

template <int S>
__global__ void __launch_bounds__(GramCfg<S>::NW * 32, (S == 1) ? 4 : 2)
gram_kernel(int64_t n, const double* __restrict__ R, const double* __restrict__ AR, const double* __restrict__ AP,
            const double* __restrict__ r, double* __restrict__ partials, ScgState* __restrict__ st, int do_solve) {
    using Cfg = GramCfg<S>;
    constexpr int G = Cfg::G, NSL = Cfg::NSL, RG = Cfg::RG;
    pdl_wait();  // (common.cuh: the predecessor in the graph may still be draining)
    pdl_launch();
    if (st->status != SCG_RUNNING) return;
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
        // all loads of the row first, as one batch (asm volatile keeps them ahead of the FMAs: memory-level parallelism
        // is what this kernel lives on).  With one slice (S <= 4) nothing is re-read, so the loads bypass L1.
        double Rv[S], ARv[G], APv[G], Rsel[G];
#pragma unroll
        for (int j = 0; j < S; j++) Rv[j] = (NSL == 1) ? ldg_stream(R + (int64_t)j * n + row) : ldg_nc(R + (int64_t)j * n + row);
#pragma unroll
        for (int g = 0; g < G; g++) {
            const bool ok = (G * NSL == S) || (c0 + g < S);
            ARv[g] = ok ? ldg_stream(AR + (int64_t)(c0 + g) * n + row) : 0.0;
            APv[g] = ok ? ldg_stream(AP + row * S + c0 + g) : 0.0;
            if constexpr (NSL == 1) Rsel[g] = Rv[g];
            else Rsel[g] = ok ? ldg_nc(R + (int64_t)(c0 + g) * n + row) : 0.0;  // R_{c0+g} again (L1 hit): keeps Rv[] statically indexed
        }
        const double rv = ldg_stream(r + row);
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
    // ---- block reduction: shuffle tree inside the warp (slice q = warp % NSL, row group rg = warp / NSL) ----
    // (all 2SG+G sums of the warp in one recursive-halving reduction: 37 shuffle steps instead of 180 at S = 4 -- these run at
    // the end of every block, when nothing overlaps them)
    __shared__ double red[Cfg::NW][Cfg::NACC];
    {
        double v[Cfg::NACC];
#pragma unroll
        for (int g = 0; g < G; g++) {
#pragma unroll
            for (int i = 0; i < S; i++) { v[i * G + g] = accM[i][g]; v[S * G + g * S + i] = accC[g][i]; }
            v[2 * S * G + g] = accm[g];
        }
        int nv;
        const int base = warp_reduce_many<Cfg::NACC>(v, lane, nv);
        constexpr int KF = warp_reduce_many_count(Cfg::NACC);
#pragma unroll
        for (int t = 0; t < KF; t++)
            if (t < nv) red[warp][base + t] = v[t];
    }
    gram_cross_block_finish<S, G, NSL, RG>(red, partials, st, do_solve);
}

// stand-alone a3 for the test hooks: same device function, operands in global memory.  Lprev != NULL: the carried-factor
// path of the solver loop (Lprev = Cholesky factor of the previous W; Wprev is then not read); Lout (may be NULL)
// receives the factor of the new W.
__global__ void small_solve_kernel(int s, const double* M, const double* C, const double* m, const double* Wprev,
                                   const double* Lprev, double* beta, double* alpha, double* W, double* Lout, int* status_out) {
    __shared__ SmallSolveSmem ssm;
    if (Lprev) {
        for (int e = threadIdx.x; e < s * s; e += 32) ssm.L[e] = Lprev[e];
        __syncwarp();
    }
    const int rc = warp_small_solve(s, M, C, m, Wprev, beta, alpha, W, ssm, threadIdx.x, Lprev != nullptr);
    if (Lout && rc == 0)
        for (int e = threadIdx.x; e < s * s; e += 32) Lout[e] = ssm.L[e];
    if (threadIdx.x == 0) status_out[0] = rc;
}

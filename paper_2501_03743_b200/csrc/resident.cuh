// resident.cuh -- SURVEY.md 8(f) NEXT-3 / H8: the WHOLE outer-iteration loop of Alg. 3 in ONE cooperative
// launch, for problems small enough that the launch latency of the s + 2 graph nodes dominates (config 1: 13 MB per
// outer iteration, 2-3 us of HBM time against ~19 us of launches).
//
// One CTA per SM owns a contiguous block of RPB rows for the whole solve and keeps everything that belongs to those
// rows on chip: its slice of the CSR arrays, dinv, x, r and the four n x s blocks R, AR, P, AP live in shared memory.
// Only the basis vectors R_j (the gather sources of the next SpMV) also go to global memory (L2), because rows of
// other CTAs read them.  One outer iteration is then
//   a1  s x [ SpMV phase (gather R_j from L2 with ld.cg, CSR slice from shared memory, Jacobi / Chebyshev epilogue),
//             grid barrier ]                                   (Alg. 4; no barrier after the last one)
//   a2  per-CTA partial sums of M = R^T AR, C = AP^T R, m = R^T r -> partials[entry][cta]; grid barrier;
//       EVERY CTA sums all partials in the same fixed order (bitwise identical in all CTAs)   (Eq. 3-4)
//   a3  every CTA runs the s x s Cholesky solves in one warp (warp_small_solve)
//   a4  block updates of the CTA's rows (Alg. 3 l.17-21), R_1 = D^-1 r -> shared + global, ||r||^2 partial;
//       grid barrier; every CTA sums the partials and takes the same stop decision            (Alg. 3 l.31-33)
// i.e. s + 1 grid barriers and no kernel boundary per outer iteration.  Measured on config 1 (32^3, s = 2): 12.1 us per
// outer iteration against 20.5 us for the graph path; per phase (CTA 0, %globaltimer): SpMV 0.7 us each, a grid barrier
// 1.8 us, Gram partials 0.9, reading the partials 1.4, the solves 1.8, update 0.6, ||r||^2 0.9 -- what is left is L2
// round trips, not bandwidth.  (Letting only the last CTA to arrive reduce + solve and publish beta, alpha was measured
// slower: 13.4 us -- it serialises arrival, reduction, solve and release.)  For s > 4 the redundant reduction of the
// 2s^2+s partials and the longer solves eat the gain, so the automatic choice is limited to s <= 4.  The state (x, r, P, AP, W, k, rho, status)
// is loaded from / stored to the same global buffers the graph path uses, so solve_begin / iterate / solve_end and
// every status code behave the same.  Arithmetic per row is the same as in spmv.cuh / gram.cuh / update.cuh.
#pragma once
#include "common.cuh"
#include "gram.cuh"
#include "small_solve.cuh"

struct ResidentParams {
    int n, rpb, nzcap, kmax, basis;
    const int* rp;
    const int* ci;
    const double* va;
    const double* dinv;
    double* Rg;        // n x s column-major: R_j, written for the gathers of other CTAs
    double* ARg;       // n x s column-major: AR of the last iteration, stored at exit (read_state hook)
    double* P;         // n x s interleaved (global copy of the state, loaded at entry / stored at exit)
    double* AP;
    double* x;
    double* r;
    double* partials;  // [2s^2+s][grid] Gram partials, then [grid] ||r||^2 partials
    ScgState* st;
};

// Grid-wide barrier of a cooperative launch.  Arrivals are counted with one atomic per CTA; the CTA that completes
// generation `gen` publishes it in a flag word of another cache line, which the others poll (so the polls do not queue
// behind the atomics at the L2 slice of the counter).  Both words are zeroed by the host before the launch.
__device__ __forceinline__ void resident_grid_barrier(ScgState* st, unsigned int& gen) {
    __syncthreads();  // the CTA's global writes of this phase happen-before thread 0's release below (cumulativity)
    gen++;
    if (threadIdx.x == 0) {
        unsigned int old, v;
        asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 1;" : "=r"(old) : "l"(&st->grid_bar) : "memory");
        if (old + 1 == gen * gridDim.x) {
            asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(&st->grid_flag), "r"(gen) : "memory");
        } else {
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(&st->grid_flag) : "memory");
            } while (v < gen);
        }
    }
    __syncthreads();
}

constexpr size_t resident_smem_bytes(int s, int rpb, int nzcap) {
    return (size_t)8 * rpb * (4 * s + 3) + (size_t)12 * nzcap + (size_t)4 * (rpb + 4) + 64;
}

template <int S>
__global__ void __launch_bounds__(512, 1) resident_kernel(const ResidentParams p) {
    constexpr int G = (S <= 3) ? S : 2;          // Gram column slice per pass (register accumulators 2*S*G + G)
    constexpr int NSL = (S + G - 1) / G;
    constexpr int NACC = 2 * S * G + G, NE = 2 * S * S + S;
    ScgState* __restrict__ st = p.st;
    if (p.kmax <= 0 || st->status != SCG_RUNNING) return;  // uniform over the grid: status is only written after a barrier

    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int RPB = p.rpb, n = p.n;
    double* sR = reinterpret_cast<double*>(smem_raw);  // [S][RPB]
    double* sAR = sR + (size_t)S * RPB;
    double* sP = sAR + (size_t)S * RPB;
    double* sAP = sP + (size_t)S * RPB;
    double* sx = sAP + (size_t)S * RPB;
    double* sr = sx + RPB;
    double* sdinv = sr + RPB;
    double* svals = sdinv + RPB;
    int* scols = reinterpret_cast<int*>(svals + p.nzcap);
    int* srp = scols + p.nzcap;  // [RPB + 1] offsets into the slice

    __shared__ double red[16][NACC];
    __shared__ double fin[NE];
    __shared__ __align__(16) double sW[S * S], sbeta[S * S];
    __shared__ double salpha[S];
    __shared__ SmallSolveSmem ssm;
    __shared__ int s_rc;
    __shared__ double s_rho;

    const int tid = threadIdx.x, bd = blockDim.x, warp = tid >> 5, lane = tid & 31, nwarps = bd >> 5;
    const int grid = gridDim.x, bid = blockIdx.x;
    const int row0 = bid * RPB;
    const int nrows = min(RPB, n - row0);

    // ---- entry: CSR slice and state of the CTA's rows -> shared memory
    const int nz0 = p.rp[row0], nz1 = p.rp[row0 + nrows];
    for (int k = nz0 + tid; k < nz1; k += bd) {
        svals[k - nz0] = p.va[k];
        scols[k - nz0] = p.ci[k];
    }
    for (int lr = tid; lr <= nrows; lr += bd) srp[lr] = p.rp[row0 + lr] - nz0;
    for (int lr = tid; lr < nrows; lr += bd) {
        const int row = row0 + lr;
        sx[lr] = p.x[row];
        sr[lr] = p.r[row];
        sdinv[lr] = p.dinv[row];
        sR[lr] = __ldcg(p.Rg + row);
#pragma unroll
        for (int j = 0; j < S; j++) {
            sP[j * RPB + lr] = p.P[(size_t)row * S + j];
            sAP[j * RPB + lr] = p.AP[(size_t)row * S + j];
        }
    }
    for (int e = tid; e < S * S; e += bd) { sW[e] = st->W[e]; sbeta[e] = st->beta[e]; ssm.L[e] = st->Lw[e]; }
    if (tid < S) salpha[tid] = st->alpha[tid];
    int k_outer = st->k;
    const double rho0 = st->rho0, rtol = st->rtol;
    double rho = st->rho;
    int status = SCG_RUNNING;
    unsigned int gen = 0;
    __syncthreads();

    // A thread owns the rows lr = tid, tid + bd, ... in every phase, so the per-row shared-memory entries need no
    // barrier between phases; barriers are only needed around the cross-thread reductions.
    for (int it = 0; it < p.kmax; it++) {
        // ------------------------------------------------------------------ a1: matrix-powers kernel (Alg. 4)
#pragma unroll 1
        for (int j = 0; j < S; j++) {
            const double* __restrict__ xg = p.Rg + (size_t)j * n;
            const bool jac = (j + 1 < S);
            const int mode = (p.basis == 0) ? 0 : (j == 0 ? 1 : 2);
            for (int lr = tid; lr < nrows; lr += bd) {
                const int lo = srp[lr], hi = srp[lr + 1];
                int c[8];
                double v[8], xv[8];
#pragma unroll
                for (int u = 0; u < 8; u++) {
                    const bool ok = lo + u < hi;
                    c[u] = ok ? scols[lo + u] : -1;
                    v[u] = ok ? svals[lo + u] : 0.0;
                }
#pragma unroll
                for (int u = 0; u < 8; u++) xv[u] = (c[u] >= 0) ? __ldcg(xg + c[u]) : 0.0;
                double acc = 0.0;
#pragma unroll
                for (int u = 0; u < 8; u++) acc = fma(v[u], xv[u], acc);
                for (int k = lo + 8; k < hi; k++) acc = fma(svals[k], __ldcg(xg + scols[k]), acc);
                sAR[j * RPB + lr] = acc;
                if (jac) {
                    double z = sdinv[lr] * acc;
                    if (mode == 1) z = z - sR[j * RPB + lr];
                    else if (mode == 2) z = 2.0 * (z - sR[j * RPB + lr]) - sR[(j - 1) * RPB + lr];
                    sR[(j + 1) * RPB + lr] = z;
                    __stcg(p.Rg + (size_t)(j + 1) * n + row0 + lr, z);
                }
            }
            if (jac) resident_grid_barrier(st, gen);
        }

        // ------------------------------------------------------------------ a2: Gram partials of the CTA's rows
#pragma unroll 1
        for (int q = 0; q < NSL; q++) {
            const int c0 = q * G;
            double accM[S][G], accC[G][S], accm[G];
#pragma unroll
            for (int g = 0; g < G; g++) {
                accm[g] = 0.0;
#pragma unroll
                for (int i = 0; i < S; i++) { accM[i][g] = 0.0; accC[g][i] = 0.0; }
            }
            for (int lr = tid; lr < nrows; lr += bd) {
                double Rv[S];
#pragma unroll
                for (int i = 0; i < S; i++) Rv[i] = sR[i * RPB + lr];
                const double rv = sr[lr];
#pragma unroll
                for (int g = 0; g < G; g++) {
                    const bool ok = (G * NSL == S) || (c0 + g < S);
                    const int col = ok ? c0 + g : 0;
                    const double ARv = ok ? sAR[col * RPB + lr] : 0.0;
                    const double APv = ok ? sAP[col * RPB + lr] : 0.0;
                    const double Rsel = ok ? sR[col * RPB + lr] : 0.0;
#pragma unroll
                    for (int i = 0; i < S; i++) {
                        accM[i][g] = fma(Rv[i], ARv, accM[i][g]);
                        accC[g][i] = fma(APv, Rv[i], accC[g][i]);
                    }
                    accm[g] = fma(Rsel, rv, accm[g]);
                }
            }
#pragma unroll
            for (int g = 0; g < G; g++) {
#pragma unroll
                for (int i = 0; i < S; i++) {
                    const double a = warp_sum(accM[i][g]);
                    const double b = warp_sum(accC[g][i]);
                    if (lane == 0) { red[warp][i * G + g] = a; red[warp][S * G + g * S + i] = b; }
                }
                const double cc = warp_sum(accm[g]);
                if (lane == 0) red[warp][2 * S * G + g] = cc;
            }
            __syncthreads();
            for (int a = tid; a < NACC; a += bd) {
                double v = 0.0;
                for (int w = 0; w < nwarps; w++) v += red[w][a];
                bool valid;
                const int ge = gram_entry<S, G>(q, a, valid);
                if (valid) __stcg(p.partials + (size_t)ge * grid + bid, v);
            }
            __syncthreads();
        }
        resident_grid_barrier(st, gen);

        // ------------------------------------------------------------------ a2 finish + a3: every CTA, identical bits
        for (int e = warp; e < NE; e += nwarps) {
            const double v = warp_sum_array(p.partials + (size_t)e * grid, grid, lane);
            if (lane == 0) fin[e] = v;
        }
        __syncthreads();
        if (warp == 0) {
            // (ssm.L carries the Cholesky factor of W from one outer iteration to the next: one factorisation each)
            const int rc = warp_small_solve(S, fin, fin + S * S, fin + 2 * S * S, nullptr, sbeta, salpha, sW, ssm, lane, /*have_L=*/true);
            if (lane == 0) s_rc = rc;
        }
        __syncthreads();
        if (s_rc != 0) {  // breakdown: x, r, P, AP keep the last good iterate (as in the graph path)
            status = s_rc;
            break;
        }

        // ------------------------------------------------------------------ a4: block updates of the CTA's rows
        double rho_part = 0.0;
        for (int lr = tid; lr < nrows; lr += bd) {
            double v[S], out[S];
            double xi = sx[lr], ri = sr[lr];
#pragma unroll
            for (int l = 0; l < S; l++) v[l] = sP[l * RPB + lr];
#pragma unroll
            for (int j = 0; j < S; j++) {
                double pj = sR[j * RPB + lr];
#pragma unroll
                for (int l = 0; l < S; l++) pj = fma(v[l], sbeta[l * S + j], pj);
                out[j] = pj;
                xi = fma(pj, salpha[j], xi);
            }
#pragma unroll
            for (int j = 0; j < S; j++) sP[j * RPB + lr] = out[j];
#pragma unroll
            for (int l = 0; l < S; l++) v[l] = sAP[l * RPB + lr];
#pragma unroll
            for (int j = 0; j < S; j++) {
                double pj = sAR[j * RPB + lr];
#pragma unroll
                for (int l = 0; l < S; l++) pj = fma(v[l], sbeta[l * S + j], pj);
                out[j] = pj;
                ri = fma(-pj, salpha[j], ri);
            }
#pragma unroll
            for (int j = 0; j < S; j++) sAP[j * RPB + lr] = out[j];
            sx[lr] = xi;
            sr[lr] = ri;
            const double r1 = sdinv[lr] * ri;
            sR[lr] = r1;
            __stcg(p.Rg + row0 + lr, r1);  // R_1 of the next outer iteration
            rho_part = fma(ri, ri, rho_part);
        }
        rho_part = warp_sum(rho_part);
        if (lane == 0) red[warp][0] = rho_part;
        __syncthreads();
        if (tid == 0) {
            double v = 0.0;
            for (int w = 0; w < nwarps; w++) v += red[w][0];
            __stcg(p.partials + (size_t)NE * grid + bid, v);
        }
        resident_grid_barrier(st, gen);

        // ------------------------------------------------------------------ a5: ||r||^2 and the stop test, every CTA
        if (warp == 0) {
            const double v = warp_sum_array(p.partials + (size_t)NE * grid, grid, lane);
            if (lane == 0) s_rho = v;
        }
        __syncthreads();
        rho = s_rho;
        k_outer++;
        if (!isfinite(rho)) status = 2;
        else if (sqrt(rho) < rtol * sqrt(rho0)) status = 0;
        if (status != SCG_RUNNING) break;
    }

    // ---- exit: state of the CTA's rows -> global memory
    for (int lr = tid; lr < nrows; lr += bd) {
        const int row = row0 + lr;
        p.x[row] = sx[lr];
        p.r[row] = sr[lr];
#pragma unroll
        for (int j = 0; j < S; j++) {
            p.P[(size_t)row * S + j] = sP[j * RPB + lr];
            p.AP[(size_t)row * S + j] = sAP[j * RPB + lr];
            p.ARg[(size_t)j * n + row] = sAR[j * RPB + lr];
        }
    }
    if (bid == 0) {
        __syncthreads();
        for (int e = tid; e < S * S; e += bd) {
            st->W[e] = sW[e];
            if (status != 2) st->Lw[e] = ssm.L[e];
            st->beta[e] = sbeta[e];
            st->M[e] = fin[e];
            st->C[e] = fin[S * S + e];
        }
        if (tid < S) { st->alpha[tid] = salpha[tid]; st->m[tid] = fin[2 * S * S + tid]; }
        if (tid == 0) {
            st->k = k_outer;
            st->rho = rho;
            if (status != SCG_RUNNING) st->status = status;
        }
    }
}

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
// i.e. s + 1 grid barriers and no kernel boundary per outer iteration (LL = false, option resident_sync = 1).  Measured on
// config 1 (32^3, s = 2; CTA 0, %globaltimer, -DSCG_RESIDENT_TIMING): SpMV 0.67 us each, a grid barrier 1.5-1.8 us (release
// fence + atomic arrival + flag poll), Gram partials 0.83, reading the partials back 1.3, the solves 1.3 (a chain of ~11
// dependent IEEE divisions / square roots, ~0.11 us each: fixed by the bit-exact contract), update 0.6, ||r||^2 0.9:
// 11.4 us per outer iteration against 18.8 us for the graph path -- L2 round trips, not bandwidth.
//
// Round 2 (LL = true, the default): the same loop with NO grid barrier.  Everything one CTA publishes for others travels as
// tagged 64-bit words (ll_* below) that the readers poll -- one hop costs 0.46 us between two SMs of an idle B200:
//   a1  the neighbours' rows of R_j are gathered as tagged words (a CTA waits only for the ~10 CTAs its rows touch);
//   a2  reduce-scatter + broadcast: CTA e sums the partials of Gram entry e (it alone polls them) in the fixed order and
//       pushes the sum into every CTA's private inbox; a CTA polls only its own inbox (a flat all-gather, everybody
//       polling everybody's partials, saturated the L2 slices holding those ~200 lines: 5-9 us);
//   a5  ||r||^2 of iteration k rides as one more entry of iteration k + 1's exchange: the stop test is taken one
//       matrix-powers kernel late (x, r, P, AP, the iteration count and the status are the same; after a converged
//       solve R(:, 2:s) and AR hold the basis of the extra kernel).
// Per phase: SpMV + exchange 1.17 us each, Gram partials 1.04, exchange of the sums 2.45 (two hops + the spread of the
// CTAs' arrival, ~1 us), solves 1.4-1.5, update 0.61 = 8.0 us per outer iteration.  Letting only the last CTA to arrive
// reduce + solve and publish beta, alpha (round 1, with barriers) was slower: 13.4 us.  For s > 4 the longer solves and
// 2s^2+s entries eat the gain, so the automatic choice is limited to s <= 4.  The state (x, r, P, AP, W, k, rho, status) is
// loaded from / stored to the same global buffers the graph path uses, so solve_begin / iterate / solve_end and every
// status code behave the same.  Arithmetic per row is the same as in spmv.cuh / gram.cuh / update.cuh; both exchange
// modes give the same bits (tests/test_gpu_resident.py).
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
    // flag-in-data exchange (LL = true instantiation; see resident_ll_* below)
    ulonglong2* llR;     // [s][n] R_j as tagged word pairs: the neighbours' gather source
    ulonglong2* llPart;  // [2 (iteration parity)][2s^2+s+1][grid] Gram partials + ||r||^2 partial of the previous iteration
    ulonglong2* llTot;   // [2][grid (destination CTA)][2s^2+s+1] the finished sums, one private inbox per CTA
    unsigned int tag0;   // tags of this launch are tag0 + 1 + iteration (the host never reuses a tag value)
};

// ---- flag-in-data ("LL") exchange between the CTAs of the resident kernel.  A published double travels as two 64-bit words,
// each = (tag << 32) | one half of the value.  A naturally aligned 64-bit scalar store is single-copy atomic, so a reader that
// finds the expected tag in a word has that half of the value of that very store: no fence, no barrier atomic, no flag line
// -- one write trip to L2 and one (polled) read trip instead of release + atomic arrival + flag poll + data read.  Tags grow
// monotonically (per launch tag0 + 1 + iteration; the host advances tag0 from launch to launch and zeroes the buffers
// before tags could wrap), so stale data can never be mistaken for new.
__device__ __forceinline__ void ll_store(ulonglong2* p, double v, unsigned int tag) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    const unsigned long long t = (unsigned long long)tag << 32;
    const unsigned long long w0 = t | (b & 0xffffffffull), w1 = t | (b >> 32);
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(w0), "l"(w1) : "memory");
}
__device__ __forceinline__ ulonglong2 ll_peek(const ulonglong2* p) {
    ulonglong2 w;
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(w.x), "=l"(w.y) : "l"(p) : "memory");
    return w;
}
__device__ __forceinline__ bool ll_ready(const ulonglong2& w, unsigned int tag) {
    return (unsigned int)(w.x >> 32) == tag && (unsigned int)(w.y >> 32) == tag;
}
__device__ __forceinline__ double ll_value(const ulonglong2& w) {
    return __longlong_as_double((long long)((w.x & 0xffffffffull) | (w.y << 32)));
}
// Polled words must not be SHARED between many CTAs: when all 148 CTAs polled the same ~200 lines of partials (a flat
// all-gather) the L2 slices holding them saturated and the stores being waited for queued behind the polls -- 5-7 us per
// all-gather, 9 us after the last store; a __nanosleep back-off made it 11 us; with the batched re-polling of ll_wait_all
// still 3.5 us against 2.45 us for the two hops of the reduce-scatter + private inboxes below.
// Every wait is bounded: a word that has not arrived after LL_SPIN_LIMIT poll rounds (tens of seconds; a healthy exchange
// takes microseconds) can only mean a broken protocol or a lost peer -- the kernel traps (the launch returns an error)
// instead of hanging the device.
constexpr unsigned int LL_SPIN_LIMIT = 1u << 26;
__device__ __forceinline__ void ll_wait(ulonglong2& w, const ulonglong2* p, unsigned int tag) {
    unsigned int spins = 0;
    while (!ll_ready(w, tag)) {
        if (++spins > LL_SPIN_LIMIT) __trap();
        w = ll_peek(p);
    }
}
// the value published at p under `tag` (waits until it has arrived)
__device__ __forceinline__ double ll_load(const ulonglong2* p, unsigned int tag) {
    ulonglong2 w = ll_peek(p);
    ll_wait(w, p, tag);
    return ll_value(w);
}
// K tagged words already peeked into w[]: re-poll ALL that have not arrived together, one L2 round trip (~0.46 us between
// two SMs of an idle B200) per round -- waiting for them one after the other costs a round trip per stale word.
template <int K, class PtrOf>
__device__ __forceinline__ void ll_wait_all(ulonglong2 (&w)[K], PtrOf ptr_of, unsigned int valid, unsigned int tag) {
    for (unsigned int spins = 0;; spins++) {
        unsigned int pend = 0;
#pragma unroll
        for (int k = 0; k < K; k++)
            if (((valid >> k) & 1u) && !ll_ready(w[k], tag)) pend |= 1u << k;
        if (!pend) return;
        if (spins > LL_SPIN_LIMIT) __trap();
#pragma unroll
        for (int k = 0; k < K; k++)
            if ((pend >> k) & 1u) w[k] = ll_peek(ptr_of(k));
    }
}

// warp_sum_array over tagged entries: the same fixed order (bit for bit the sum warp_sum_array would give on plain doubles)
__device__ __forceinline__ double warp_sum_ll(const ulonglong2* p, int cnt, int lane, unsigned int tag) {
    double a[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (int b = lane;; b += 256) {  // warp_sum_array's full batches, then its predicated tail batch
        ulonglong2 w[8];
        unsigned int valid = 0;
#pragma unroll
        for (int k = 0; k < 8; k++)
            if (b + 32 * k < cnt) { w[k] = ll_peek(p + b + 32 * k); valid |= 1u << k; }
        ll_wait_all<8>(w, [&](int k) { return p + b + 32 * k; }, valid, tag);
#pragma unroll
        for (int k = 0; k < 8; k++) a[k] += ((valid >> k) & 1u) ? ll_value(w[k]) : 0.0;
        if (b + 224 >= cnt) break;
    }
    double v = ((a[0] + a[1]) + (a[2] + a[3])) + ((a[4] + a[5]) + (a[6] + a[7]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Profiling aid, compiled in only with -DSCG_RESIDENT_TIMING (never in the product build): thread 0 of CTA 0 accumulates the
// %globaltimer time between phase boundaries and prints the per-iteration means when the kernel ends.
#ifdef SCG_RESIDENT_TIMING
#define SCG_STAMP(i)                                                            \
    do {                                                                        \
        if (bid == 0 && tid == 0) {                                             \
            unsigned long long t_;                                              \
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));              \
            t_acc[i] += (double)(t_ - t_last);                                  \
            t_last = t_;                                                        \
        }                                                                       \
    } while (0)
#else
#define SCG_STAMP(i) do { } while (0)
#endif

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

// LL = false: s + 1 grid barriers per outer iteration (round 1).  LL = true (round 2, default): no grid barrier at all --
// R_j travels to the neighbours' gathers and the Gram partials to everybody as tagged words (ll_* above), and ||r||^2 of
// iteration k rides in the Gram all-gather of iteration k + 1, so the stop test is taken one matrix-powers kernel late
// (a converged solve computes one MPK more; x, r, P, AP and the iteration count are the same).
template <int S, bool LL>
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
    __shared__ double fin[NE + 1];  // (LL: entry NE = ||r||^2 of the previous iteration)
    __shared__ double s_rho_cta;    // LL: this CTA's ||r||^2 partial of the last update, published with the next Gram partials
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
    if (LL) {  // publish the CTA's rows of R_1 for the neighbours' first gathers
        for (int lr = tid; lr < nrows; lr += bd) ll_store(p.llR + row0 + lr, sR[lr], p.tag0 + 1u);
        if (tid == 0) s_rho_cta = 0.0;
    }
    __syncthreads();
    if (S <= 2 && warp == 0) warp_prepare_divisors(S, ssm.L, ssm.Rd, lane);  // (for thread_small_solve below, which keeps them in step with ssm.L)

    // A thread owns the rows lr = tid, tid + bd, ... in every phase, so the per-row shared-memory entries need no
    // barrier between phases; barriers are only needed around the cross-thread reductions.
#ifdef SCG_RESIDENT_TIMING
    double t_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    unsigned long long t_last = 0;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_last));
#endif
    for (int it = 0; it < p.kmax; it++) {
        SCG_STAMP(0);
        const unsigned int tag = p.tag0 + 1u + (unsigned int)it;  // LL: everything published for this iteration carries it
        // ------------------------------------------------------------------ a1: matrix-powers kernel (Alg. 4)
#pragma unroll 1
        for (int j = 0; j < S; j++) {
            const double* __restrict__ xg = p.Rg + (size_t)j * n;
            const ulonglong2* xl = p.llR + (size_t)j * n;
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
                if (LL) {  // all eight tagged loads in flight, then whatever has not arrived yet is polled
                    // (taking the CTA's own rows from shared memory instead was measured: no gain -- every row of a 3-D stencil
                    // has neighbours in other CTAs and waits one hop for them anyway)
                    ulonglong2 w[8];
                    unsigned int valid = 0;
#pragma unroll
                    for (int u = 0; u < 8; u++)
                        if (c[u] >= 0) { w[u] = ll_peek(xl + c[u]); valid |= 1u << u; }
                    ll_wait_all<8>(w, [&](int u) { return xl + c[u]; }, valid, tag);
#pragma unroll
                    for (int u = 0; u < 8; u++) xv[u] = ((valid >> u) & 1u) ? ll_value(w[u]) : 0.0;
                } else {
#pragma unroll
                    for (int u = 0; u < 8; u++) xv[u] = (c[u] >= 0) ? __ldcg(xg + c[u]) : 0.0;
                }
                double acc = 0.0;
#pragma unroll
                for (int u = 0; u < 8; u++) acc = fma(v[u], xv[u], acc);
                for (int k = lo + 8; k < hi; k++) acc = fma(svals[k], LL ? ll_load(xl + scols[k], tag) : __ldcg(xg + scols[k]), acc);
                sAR[j * RPB + lr] = acc;
                if (jac) {
                    double z = sdinv[lr] * acc;
                    if (mode == 1) z = z - sR[j * RPB + lr];
                    else if (mode == 2) z = 2.0 * (z - sR[j * RPB + lr]) - sR[(j - 1) * RPB + lr];
                    sR[(j + 1) * RPB + lr] = z;
                    if (LL) ll_store(p.llR + (size_t)(j + 1) * n + row0 + lr, z, tag);
                    else __stcg(p.Rg + (size_t)(j + 1) * n + row0 + lr, z);
                }
            }
            if (jac && !LL) resident_grid_barrier(st, gen);
            if (j == 0) SCG_STAMP(1);
        }
        SCG_STAMP(2);

        // ------------------------------------------------------------------ a2: Gram partials of the CTA's rows
        ulonglong2* part = p.llPart + (size_t)(it & 1) * (NE + 1) * grid;  // LL: two slots by iteration parity (a CTA can be at
        // most one all-gather ahead of the slowest reader: it cannot publish iteration it + 1 before everybody published it)
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
            {  // all sums of the warp in one recursive-halving reduction (common.cuh)
                double v[NACC];
#pragma unroll
                for (int g = 0; g < G; g++) {
#pragma unroll
                    for (int i = 0; i < S; i++) { v[i * G + g] = accM[i][g]; v[S * G + g * S + i] = accC[g][i]; }
                    v[2 * S * G + g] = accm[g];
                }
                int nv;
                const int base = warp_reduce_many<NACC>(v, lane, nv);
                constexpr int KF = warp_reduce_many_count(NACC);
#pragma unroll
                for (int t = 0; t < KF; t++)
                    if (t < nv) red[warp][base + t] = v[t];
            }
            __syncthreads();
            for (int a = tid; a < NACC; a += bd) {
                double v = 0.0;
                for (int w = 0; w < nwarps; w++) v += red[w][a];
                bool valid;
                const int ge = gram_entry<S, G>(q, a, valid);
                if (valid) {
                    if (LL) ll_store(part + (size_t)ge * grid + bid, v, tag);
                    else __stcg(p.partials + (size_t)ge * grid + bid, v);
                }
            }
            __syncthreads();
        }
        SCG_STAMP(3);
#ifdef SCG_RESIDENT_TIMING
        if (LL && it == 10 && tid == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); p.partials[bid] = (double)(t_ % 1000000000ull); }
#endif
        if (LL) {
            if (tid == 0) ll_store(part + (size_t)NE * grid + bid, s_rho_cta, tag);
        } else {
            resident_grid_barrier(st, gen);
        }

        // ------------------------------------------------------------------ a2 finish + a3: every CTA, identical bits
        if (LL) {
            // reduce-scatter + broadcast: entry e is summed (fixed order) by ONE warp of CTA e % grid, the only poller of
            // that entry's partials, which pushes the sum into every CTA's private inbox; a CTA polls only its own inbox
            ulonglong2* tot = p.llTot + (size_t)(it & 1) * grid * (NE + 1);
            for (int e = bid + warp * grid; e < NE + 1; e += nwarps * grid) {
                const double v = warp_sum_ll(part + (size_t)e * grid, grid, lane, tag);
                for (int dst = lane; dst < grid; dst += 32) ll_store(tot + (size_t)dst * (NE + 1) + e, v, tag);
            }
            for (int e = tid; e < NE + 1; e += bd) fin[e] = ll_load(tot + (size_t)bid * (NE + 1) + e, tag);
        } else {
            for (int e = warp; e < NE; e += nwarps) {
                const double v = warp_sum_array(p.partials + (size_t)e * grid, grid, lane);
                if (lane == 0) fin[e] = v;
            }
        }
        __syncthreads();
#ifdef SCG_RESIDENT_TIMING
        if (LL && it == 10 && tid == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); p.partials[grid + bid] = (double)(t_ % 1000000000ull); }
#endif
        SCG_STAMP(4);
        if (LL && it > 0) {  // a5 of the PREVIOUS iteration: ||r||^2 and the stop test, every CTA, identical bits
            rho = fin[NE];
            if (!isfinite(rho)) status = 2;
            else if (sqrt(rho) < rtol * sqrt(rho0)) status = 0;
            if (status != SCG_RUNNING) break;
        }
        if (warp == 0) {
            // (ssm.L carries the Cholesky factor of W from one outer iteration to the next: one factorisation each)
            int rc;
            if constexpr (S <= 2) {  // in registers, fully unrolled, same operations and roundings (small_solve.cuh)
                double Lc[S * S], Rc[S], be[S * S], al[S], Wn[S * S];
#pragma unroll
                for (int e = 0; e < S * S; e++) Lc[e] = ssm.L[e];
#pragma unroll
                for (int i = 0; i < S; i++) Rc[i] = ssm.Rd[i];
                rc = thread_small_solve<S>(fin, fin + S * S, fin + 2 * S * S, Lc, Rc, be, al, Wn);
                __syncwarp();  // every lane has read ssm.L / ssm.Rd
                if (lane == 0 && rc == 0) {
#pragma unroll
                    for (int e = 0; e < S * S; e++) { sbeta[e] = be[e]; sW[e] = Wn[e]; ssm.L[e] = Lc[e]; }
#pragma unroll
                    for (int i = 0; i < S; i++) { salpha[i] = al[i]; ssm.Rd[i] = Rc[i]; }
                }
            } else {
                rc = warp_small_solve(S, fin, fin + S * S, fin + 2 * S * S, nullptr, sbeta, salpha, sW, ssm, lane, /*have_L=*/true);
            }
            if (lane == 0) s_rc = rc;
        }
        __syncthreads();
        SCG_STAMP(5);
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
            if (LL) ll_store(p.llR + row0 + lr, r1, tag + 1u);  // R_1 of the next outer iteration
            else __stcg(p.Rg + row0 + lr, r1);
            rho_part = fma(ri, ri, rho_part);
        }
        rho_part = warp_sum(rho_part);
        if (lane == 0) red[warp][0] = rho_part;
        __syncthreads();
        if (tid == 0) {
            double v = 0.0;
            for (int w = 0; w < nwarps; w++) v += red[w][0];
            if (LL) s_rho_cta = v;
            else __stcg(p.partials + (size_t)NE * grid + bid, v);
        }
        if (LL) {  // (the sum over the CTAs rides in the next iteration's all-gather, or in the one after the loop)
            k_outer++;
            __syncthreads();
            SCG_STAMP(6);  // red[] is reused by the next Gram reduction; s_rho_cta is read by thread 0 only
            continue;
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
        SCG_STAMP(6);
        if (status != SCG_RUNNING) break;
    }
#ifdef SCG_RESIDENT_TIMING
    if (LL && bid == 0 && tid == 0 && p.kmax >= 20) {
        double s0 = 1e30, s1 = -1e30, d0 = 1e30, d1 = -1e30;
        int imax = 0;
        for (int b = 0; b < grid; b++) {
            const double a = __ldcg(p.partials + b), d = __ldcg(p.partials + grid + b);
            if (a < s0) s0 = a;
            if (a > s1) { s1 = a; imax = b; }
            if (d < d0) d0 = d;
            if (d > d1) d1 = d;
        }
        printf("  iteration 10: partial stores spread over %.0f ns (last: CTA %d); all-gather done %.0f .. %.0f ns after the first store, i.e. %.0f .. %.0f ns after the LAST store\n",
               s1 - s0, imax, d0 - s0, d1 - s0, d0 - s1, d1 - s1);
    }
    if (bid == 0 && tid == 0 && p.kmax >= 20)
        printf("resident LL=%d kmax=%d ns per iteration: top %.0f | spmv1(+exch) %.0f | other spmv %.0f | gram partials %.0f | allgather/barrier+sum %.0f | "
               "solve %.0f | update(+rho) %.0f\n", (int)LL, p.kmax, t_acc[0] / p.kmax, t_acc[1] / p.kmax, t_acc[2] / p.kmax, t_acc[3] / p.kmax,
               t_acc[4] / p.kmax, t_acc[5] / p.kmax, t_acc[6] / p.kmax);
#endif

    if (LL && status == SCG_RUNNING) {  // all kmax iterations done: ||r||^2 of the last one, one all-gather of its own
        const unsigned int tagf = p.tag0 + 1u + (unsigned int)p.kmax;
        ulonglong2* partf = p.llPart + (size_t)(p.kmax & 1) * (NE + 1) * grid + (size_t)NE * grid;
        __syncthreads();
        ulonglong2* totf = p.llTot + (size_t)(p.kmax & 1) * grid * (NE + 1);
        if (tid == 0) ll_store(partf + bid, s_rho_cta, tagf);
        if (bid == NE % grid && warp == 0) {  // the one reducer; everybody else polls only its own inbox
            const double v = warp_sum_ll(partf, grid, lane, tagf);
            for (int dst = lane; dst < grid; dst += 32) ll_store(totf + (size_t)dst * (NE + 1) + NE, v, tagf);
        }
        if (tid == 0) s_rho = ll_load(totf + (size_t)bid * (NE + 1) + NE, tagf);
        __syncthreads();
        rho = s_rho;
        if (!isfinite(rho)) status = 2;
        else if (sqrt(rho) < rtol * sqrt(rho0)) status = 0;
    }

    // ---- exit: state of the CTA's rows -> global memory
    if (LL)  // the basis columns in plain doubles (R_1 = D^-1 r of the next iteration first), for the next launch / read_state
        for (int lr = tid; lr < nrows; lr += bd)
#pragma unroll
            for (int j = 0; j < S; j++) p.Rg[(size_t)j * n + row0 + lr] = sR[j * RPB + lr];
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

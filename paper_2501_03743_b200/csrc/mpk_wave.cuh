// mpk_wave.cuh -- the matrix-powers kernel (Alg. 4) as ONE wavefront-ordered kernel per pass, so that
// the CSR arrays are read from HBM once per pass of `nlev` levels instead of once per level (option "mpk_fused").
//
// The s SpMVs of the MPK sweep the same matrix s times: s (12 nnz + 4n) of the (184 s + 40) n bytes of an outer
// iteration -- 57 % at s = 4 on the 7-point configs.  For a banded matrix (half bandwidth bw rows) level j+1 only needs
// level j on the rows within +-bw, so the levels can follow each other down the matrix a fixed distance apart: the rows
// of A streamed from HBM by the first level of a pass are touched again by the next levels within (nlev-1) * lag rows
// of progress -- a window of a few tens of MB that stays in the 126 MB L2 (measured on this B200: an L2-resident
// buffer of <= 64 MB streams at 18 TB/s against 7.2 TB/s from HBM).  The basis vectors R_{j+1} written by level j are
// gathered by level j+1 out of L2 as well.  This is the communication-avoiding matrix-powers idea the paper cites as
// related work applied to the cache hierarchy of one GPU instead of to the network.
//
// Round 1's version of this file assigned warp tiles statically (every warp tied to the slowest one) and staged through
// per-warp rings; it halved the DRAM traffic but lost to the separate SpMVs (820 vs 550 us per level).  This version:
//   * work ITEMS (level, block of BR = SPI * TR rows) in wavefront order  q -> t = q / nlev, lev = q % nlev,
//     block = t - lev * lag;  CTA c of a persistent grid takes the items c, c + G, c + 2G, ... (G <= occupancy * SMs, so
//     all CTAs are resident once their predecessors in the stream have drained).  Claiming items with an atomic was
//     tried first: the claim -> rowptr -> copy latency chain of the producer (three L2 round trips per item) bound the
//     kernel, and claiming ahead to hide it inflates the rows in flight, hence the lag and the L2 window;
//   * the CTA-wide producer / consumer TMA pipeline of spmv_cta.cuh (few large bulk copies in flight): the producer
//     warp stages colidx / vals / rowptr of each 256-row stage and checks the item's dependency while the copies fly
//     (the facts of the NEXT stage are fetched one stage ahead); the consumer warps compute exactly the rows of spmv_cta_kernel (same bits);
//   * dependency of (lev, b): level lev-1 complete on blocks 0 .. b + dep - 1 (dep = ceil(bw / BR) + 1).  Per-item done
//     counters (one red.release.gpu per consumer warp, issued one stage late) and a per-level watermark of leading complete
//     blocks that the WAITERS advance (scan of <= 32 flags per probe); in the schedule a level trails its predecessor by
//     lag = dep + slack blocks, the slack covering the items the grid has in flight, so a prerequisite was published
//     long before it is needed and the check is one or two relaxed loads off the critical path.
// Coherence of the gathers.  R_{j+1} is written during the kernel by other SMs and gathered through L1.  A row is read
// only after its block's flag was seen set, the writer published the flag with a gpu-scope release after its stores,
// L1 is filled per 32-byte sector and blocks start at multiples of 256 rows of a column whose base is 32-byte aligned
// (setup requires n % 4 == 0), and L1 is empty at kernel start: no sector can be in L1 from before it was final.  The
// reader side uses relaxed loads (an acquire would compile to CCTL.IVALL and drop the SM's whole L1 per item); under
// the PTX memory model that is formally a race on the gathered data -- the hardware assumption (no stale sector can
// exist, stores of a released block have reached L2) is stated here and next to the option in sstep_cg.h.
#pragma once
#include "common.cuh"
#include "spmv.cuh"

struct MpkWaveParams {
    int n, nnz, s;
    int j0, nlev;        // levels [j0, j0 + nlev) in this launch
    int nb;              // blocks of BR rows
    int lag;             // blocks a level trails the previous one by in the schedule (dep + slack)
    int dep;             // level lev on block b needs level lev-1 complete on blocks 0 .. b + dep - 1
    int bp;              // back-pressure: level 0 on block b needs the last level complete on blocks 0 .. b - (nlev-1) lag - bp - 1
    int basis;
    const int* rp;
    const int* ci;
    const double* va;
    double* R;           // n x s column-major; R(:, j0) is the input
    double* AR;
    const ScgState* st;
    int* watermark;      // [nlev * 32] leading complete blocks per level, one 128-byte line each (zeroed)
    int* done;           // [nlev][nb] consumer warps that have finished the item (zeroed); complete at NCW
};

struct MpkStageInfo {
    int row0;   // first row of the stage; -1 = no more work (consumers leave)
    int lev;    // level relative to j0
    int a0;     // first staged nnz index
    int blk;    // block of the item
    int last;   // last stage of its item
    int slot;   // item slot (completion counter)
};

__device__ __forceinline__ int ld_relaxed_gpu(const int* p) {
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

template <int D, int TR, int CAPT, int SPI>
struct MpkWaveCfg {
    static constexpr int NCW = TR / 32;
    static constexpr int THREADS = TR + 32;
    static constexpr int BR = TR * SPI;
    static constexpr int RPW = TR + 4;                       // staged rowptr entries per stage (TR + 1, padded to 16 bytes)
    static constexpr size_t STAGE = (size_t)CAPT * 12 + (size_t)RPW * 4;
    static constexpr size_t SMEM = (size_t)D * STAGE + (size_t)D * 16 + (size_t)D * sizeof(MpkStageInfo) + 64;
};

// XOPT: experiment switches (0 in the product): 1 = evict-first hint on every level, 2 = plain (not streaming) AR stores,
// 4 = rowptr of the stage by plain loads instead of a bulk copy, 8 = no completion signals, 16 = no dependency waits (8, 16: timing only)
template <int D, int TR, int CAPT, int SPI, int XOPT = 0>
__global__ void __launch_bounds__(TR + 32, 3) mpk_wave_kernel(const MpkWaveParams p) {
    using Cfg = MpkWaveCfg<D, TR, CAPT, SPI>;
    constexpr int NCW = Cfg::NCW, U = 8, RPW = Cfg::RPW, BR = Cfg::BR, NSLOT = 4;
    pdl_wait();
    pdl_launch();
    if (p.st && p.st->status != SCG_RUNNING) return;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* svals = reinterpret_cast<double*>(smem_raw);                                  // [D][CAPT]
    int* scols = reinterpret_cast<int*>(smem_raw + (size_t)D * CAPT * 8);                 // [D][CAPT]
    int* srp = reinterpret_cast<int*>(smem_raw + (size_t)D * CAPT * 12);                  // [D][RPW]
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)D * Cfg::STAGE);
    uint64_t* empty = full + D;
    MpkStageInfo* info = reinterpret_cast<MpkStageInfo*>(empty + D);
    int* s_cnt = reinterpret_cast<int*>(info + D);                                        // [NSLOT] consumer warps done per item slot
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = p.n, nnz = p.nnz, NB = p.nb, nlev = p.nlev;

    if (threadIdx.x == 0) {
#pragma unroll
        for (int d = 0; d < D; d++) { mbar_init(&full[d], 2); mbar_init(&empty[d], NCW); }  // full: copies armed + dependency met
        mbar_fence_init();
    }
    if (threadIdx.x < NSLOT) s_cnt[threadIdx.x] = 0;
    __syncthreads();

    if (warp == NCW) {
        // ------------------------------------------------------------------ producer warp: stage, check dependencies
        // The CTA's items are q = blockIdx.x, blockIdx.x + gridDim.x, ... of the wavefront sequence, so everything about the
        // next stage (its rowptr ends, the watermark it depends on) is fetched while the current one is being staged: the
        // producer pays one L2 round trip per stage, overlapped with its wait for a free slot.
        const uint64_t pol_last = l2_policy_evict_first();
        const int total = (NB + (nlev - 1) * p.lag) * nlev;  // setup guarantees < 2^31
        const int G = (int)gridDim.x;
        int wm_seen[5] = {0, 0, 0, 0, 0};  // last watermark seen per level (nlev <= 5)
        // candidate stage kk -> (item, stage inside the item); returns false when the CTA's sequence is exhausted
        struct Cand { int lev, blk, row0, first; };
        int kk = 0;
        auto next_valid = [&](Cand& c) -> bool {
            for (;; kk++) {
                const int it = kk / SPI, sp = kk - it * SPI;
                // (the CTA's position rotates from round to round, so that every CTA takes items of every level: the grid size
                // is a multiple of nlev more often than not)
                const long long q = (long long)it * G + (long long)(((int)blockIdx.x + it) % G);
                if (q >= total) return false;
                const int t = (int)(q / nlev), lev = (int)(q - (long long)t * nlev);
                const int blk = t - lev * p.lag;
                if (blk < 0 || blk >= NB) { kk += SPI - 1 - sp; continue; }
                const int row0 = blk * BR + sp * TR;
                if (row0 >= n) continue;
                c.lev = lev; c.blk = blk; c.row0 = row0; c.first = (sp == 0);
                kk++;
                return true;
            }
        };
        // prefetched facts of a stage: nnz range (lanes 0, 1 load rowptr) and the watermark of its prerequisite level (lane 2)
        auto prefetch = [&](const Cand& c, int& v) {
            v = 0;
            int row1 = c.row0 + TR;
            if (row1 > n) row1 = n;
            if (lane == 0) v = p.rp[c.row0];
            else if (lane == 1) v = p.rp[row1];
            else if (lane == 2 && c.first && nlev > 1)
                v = ld_relaxed_gpu(p.watermark + (size_t)(c.lev > 0 ? c.lev - 1 : nlev - 1) * 32);
        };
        Cand cur, nxt;
        int pv_cur = 0, pv_nxt = 0;
        bool have = next_valid(cur);
        if (have) prefetch(cur, pv_cur);
        int k = 0;       // stages issued by this CTA
        int items = 0;   // items started by this CTA
        while (have) {
            const bool have_next = next_valid(nxt);
            if (have_next) prefetch(nxt, pv_nxt);   // in flight while this stage is staged
            const int lev = cur.lev, blk = cur.blk, row0 = cur.row0;
            if (cur.first) items++;
            const int slot = (items - 1) % NSLOT;
            const bool last_level = (XOPT & 1) || (p.j0 + lev + 1 == p.s) || (lev + 1 == nlev);
            const int sl = k % D;
            if (k >= D) mbar_wait(&empty[sl], (uint32_t)(((k / D) - 1) & 1));
            int row1 = row0 + TR;
            if (row1 > n) row1 = n;
            const int nz0 = __shfl_sync(0xffffffffu, pv_cur, 0);
            const int nz1 = __shfl_sync(0xffffffffu, pv_cur, 1);
            const int wm_pre = __shfl_sync(0xffffffffu, pv_cur, 2);
            const int a0 = nz0 & ~3;
            int bulk_end = (nz1 + 3) & ~3;
            const int lim = nnz & ~3;
            if (bulk_end > lim) bulk_end = lim;
            if (bulk_end < a0) bulk_end = a0;
            const int cnt = bulk_end - a0;
            double* dv = svals + (size_t)sl * CAPT;
            int* dc = scols + (size_t)sl * CAPT;
            int* dr = srp + (size_t)sl * RPW;
            for (int e = bulk_end + lane; e < nz1; e += 32) { dv[e - a0] = p.va[e]; dc[e - a0] = p.ci[e]; }
            // rowptr of the stage: one bulk copy of RPW entries, or plain loads where that would run past rowptr[n]
            const bool rp_bulk = !(XOPT & 4) && (row0 + RPW <= n + 1);
            if (!rp_bulk)
                for (int e = lane; e <= row1 - row0; e += 32) dr[e] = p.rp[row0 + e];
            if (lane == 0) {
                MpkStageInfo si;
                si.row0 = row0; si.lev = lev; si.a0 = a0; si.blk = blk; si.slot = slot;
                si.last = ((row0 - blk * BR) / TR + 1 == SPI || row0 + TR >= n) ? 1 : 0;
                info[sl] = si;
            }
            __syncwarp();
            if (lane == 0) {
                fence_proxy_async_smem();
                const uint32_t bytes = (uint32_t)cnt * 12u + (rp_bulk ? (uint32_t)RPW * 4u : 0u);
                if (bytes > 0) {
                    mbar_expect_tx(&full[sl], bytes);
                    if (cnt > 0) {
                        if (last_level) {
                            bulk_g2s(dv, p.va + a0, (uint32_t)cnt * 8u, &full[sl], pol_last);
                            bulk_g2s(dc, p.ci + a0, (uint32_t)cnt * 4u, &full[sl], pol_last);
                        } else {  // default L2 policy: the slice is re-read by the next level of the pass
                            bulk_g2s_nohint(dv, p.va + a0, (uint32_t)cnt * 8u, &full[sl]);
                            bulk_g2s_nohint(dc, p.ci + a0, (uint32_t)cnt * 4u, &full[sl]);
                        }
                    }
                    if (rp_bulk) bulk_g2s_nohint(dr, p.rp + row0, (uint32_t)RPW * 4u, &full[sl]);
                } else {
                    mbar_arrive(&full[sl]);
                }
            }
            // dependencies of the item, checked at its first stage while the copies are in flight:
            //   lev > 0 : level lev-1 complete on the first blk + dep blocks (the rows this block gathers from);
            //   lev = 0 : back-pressure -- the LAST level of the pass complete up to `bp` blocks behind, so that the first level
            //             (which waits for nobody) cannot run away from the others and blow the L2 window
            if (cur.first && nlev > 1 && !(XOPT & 16)) {
                const int wl = (lev > 0) ? lev - 1 : nlev - 1;
                int need = (lev > 0) ? blk + p.dep : blk - (nlev - 1) * p.lag - p.bp;
                if (need > NB) need = NB;
                int seen = 0;
#pragma unroll
                for (int l = 0; l < 5; l++)
                    if (l == wl) seen = wm_seen[l];
                if (seen < wm_pre) seen = wm_pre;
                if (seen < need) {
                    const int* flags = p.done + (size_t)wl * NB;
                    int w = seen;
                    unsigned ns = 32;
                    while (w < need) {  // advance over leading set flags, 32 per probe
                        const int bq = w + lane;
                        const int f = (bq < NB) ? ld_relaxed_gpu(flags + bq) : 0;
                        const unsigned m = __ballot_sync(0xffffffffu, f >= NCW);
                        const int lead = (m == 0xffffffffu) ? 32 : (__ffs(~m) - 1);
                        w += lead;
                        if (w > NB) w = NB;
                        if (lead < 32 && w < need) {
                            __nanosleep(ns);
                            if (ns < 512) ns *= 2;
                        }
                    }
                    if (lane == 0) atomicMax(p.watermark + (size_t)wl * 32, w);
                    seen = w;
                }
#pragma unroll
                for (int l = 0; l < 5; l++)
                    if (l == wl) wm_seen[l] = seen;
            }
            if (lane == 0) mbar_arrive(&full[sl]);  // second arrival: the stage may be consumed
            k++;
            cur = nxt;
            pv_cur = pv_nxt;
            have = have_next;
        }
        // sentinel stage: the consumers leave
        {
            const int sl = k % D;
            if (k >= D) mbar_wait(&empty[sl], (uint32_t)(((k / D) - 1) & 1));
            if (lane == 0) {
                info[sl].row0 = -1;
                mbar_arrive(&full[sl]);
                mbar_arrive(&full[sl]);
            }
        }
        return;
    }

    // ---------------------------------------------------------------------- consumer warps
    // Completion of an item is signalled per warp and ONE STAGE LATE: a release (MEMBAR + red) right after the stores would
    // stall the warp for a full write round trip; issued behind the next stage's gathers it waits for nothing the warp
    // would not wait for anyway.  An item is complete when all NCW warps have counted it.
    int* pend = nullptr;
    auto signal_pending = [&]() {
        if (pend) {
            __syncwarp();  // the lanes' stores are ordered before lane 0's release (cumulativity)
            if (lane == 0) asm volatile("red.release.gpu.global.add.s32 [%0], 1;" ::"l"(pend) : "memory");
            pend = nullptr;
        }
    };
    for (int k = 0;; k++) {
        const int sl = k % D;
        if (pend && !mbar_test(&full[sl], (uint32_t)((k / D) & 1))) signal_pending();  // never block holding an unsignalled item:
        mbar_wait(&full[sl], (uint32_t)((k / D) & 1));                                 // the stage may be waiting for exactly it
        const MpkStageInfo si = info[sl];
        if (si.row0 < 0) break;
        const int j = p.j0 + si.lev;
        const int lr = warp * 32 + lane;
        const int row = si.row0 + lr;
        const bool live = row < n;
        const double* __restrict__ x = p.R + (size_t)j * n;
        const int* dr = srp + (size_t)sl * RPW;
        int lo = 0, hi = 0;
        if (live) { lo = dr[lr]; hi = dr[lr + 1]; }
        const double* sv = svals + (size_t)sl * CAPT - si.a0;
        const int* sc = scols + (size_t)sl * CAPT - si.a0;
        int c[U];
        double v[U], xv[U];
        double diag = 0.0;
#pragma unroll
        for (int u = 0; u < U; u++) {
            const int kk = lo + u;
            const bool ok = kk < hi;
            c[u] = ok ? sc[kk] : -1;
            v[u] = ok ? sv[kk] : 0.0;
            if (c[u] == row) diag = v[u];
        }
#pragma unroll
        for (int u = 0; u < U; u++) xv[u] = (c[u] >= 0) ? x[c[u]] : 0.0;
        signal_pending();  // the previous item's completion, behind this stage's gathers
        const bool jac = (j + 1 < p.s);
        const int mode = (p.basis == 0) ? 0 : (j == 0 ? 1 : 2);
        double xrow = 0.0, xpv = 0.0;
        if (jac && mode != 0 && live) {
            xrow = x[row];
            if (mode == 2) xpv = p.R[(size_t)(j - 1) * n + row];
        }
        double rem = 0.0;
        for (int k0 = lo + U; k0 < hi; k0 += U) {  // rows longer than U entries
            int cc[U];
            double vv[U], xx[U];
#pragma unroll
            for (int u = 0; u < U; u++) {
                const int kk = k0 + u;
                const bool ok = kk < hi;
                cc[u] = ok ? sc[kk] : -1;
                vv[u] = ok ? sv[kk] : 0.0;
                if (cc[u] == row) diag = vv[u];
            }
#pragma unroll
            for (int u = 0; u < U; u++) xx[u] = (cc[u] >= 0) ? x[cc[u]] : 0.0;
#pragma unroll
            for (int u = 0; u < U; u++) rem = fma(vv[u], xx[u], rem);
        }
        __syncwarp();  // every lane has read the stage
        if (lane == 0) mbar_arrive(&empty[sl]);
        double acc = 0.0;
#pragma unroll
        for (int u = 0; u < U; u++) acc = fma(v[u], xv[u], acc);
        acc += rem;
        if (live) {
            if (XOPT & 2) p.AR[(size_t)j * n + row] = acc;
            else __stcs(p.AR + (size_t)j * n + row, acc);  // AR_j is not read again before the Gram kernel: streaming store
            if (jac) {
                double z = __drcp_rn(diag) * acc;
                if (mode == 1) z = z - xrow;
                else if (mode == 2) z = 2.0 * (z - xrow) - xpv;
                p.R[(size_t)(j + 1) * n + row] = z;
            }
        }
        if (si.last && nlev > 1 && !(XOPT & 8)) pend = p.done + (size_t)si.lev * NB + si.blk;
    }
    signal_pending();
}

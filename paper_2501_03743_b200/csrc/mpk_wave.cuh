// mpk_wave.cuh -- the matrix-powers kernel (Alg. 4) as ONE wavefront-ordered kernel, so that the CSR
// arrays are read from HBM once per outer iteration instead of s times (option "mpk_fused" = 2; EXPERIMENTAL, off by
// default).
//
// Status (B200, 7-point 256^3 / 320^3, s = 2 and 4, ncu + CUDA events): bitwise the same R, AR as the separate SpMVs;
// DRAM reads of a two-level pass 3.2 -> 1.6 GB (the second level hits L2, as designed); but 820-840 us per level
// against 550 us for spmv_bulk_kernel.  History of what it took to get there: acquire polls and __threadfence() compile
// to CCTL.IVALL (L1 dropped per poll / per tile); a worker that advanced the watermark when it completed a block became
// the straggler of the whole grid (5200 us per two levels); thousands of pollers on one address saturate its L2 slice.
// What is left: tiles are assigned to warps statically and walked in order, so every warp is tied (within the slack) to
// the slowest warp of the grid; ~25 % of the issued instructions are polls.  Also tried: one warp group per level (level 0
// then never waits for anybody) -- 1360 us per level: with the warps split between the levels each level is bound by
// the per-tile latency of its half of the warps (24 warps per SM is what 80 registers and the staging ring allow).
// Next step: dynamic (chunked, atomically claimed) tile assignment, so that slow warps simply take fewer tiles, and a
// leaner tile (fewer registers, more resident warps).
//
// The s SpMVs of the MPK sweep the same matrix s times: s (12 nnz + 4n) of the (184 s + 40) n bytes of an outer
// iteration.  For a banded matrix (half bandwidth bw rows) level j+1 of the MPK only needs level j on the rows within
// +-bw, so the levels can follow each other down the matrix a few row blocks apart: the rows of A touched by level 0 are
// touched again by level 1, 2, ... within (s-1) * lag * B rows of progress -- a window of a few tens of MB that stays
// in the 126 MB L2.  The vectors R_{j+1} written by level j are gathered by level j+1 out of L2 as well.  (This is the
// communication-avoiding matrix-powers idea the paper cites as related work, applied to the cache
// hierarchy of one GPU instead of to the network.)
//
// Schedule.  Rows are cut into blocks of B rows (TPB = B/32 warp tiles).  The global tile sequence is
//     q -> step t = q / (nlev * TPB),  level j = j0 + (q / TPB) % nlev,  block i = t - (j - j0) * lag,  tile q % TPB
// (tiles whose block falls outside [0, NB) are empty).  Warps of a persistent grid take the tiles q = gw, gw + GW, ...
// in order -- the same per-warp TMA ring as spmv_bulk_kernel streams colidx / vals into shared memory ahead of use.
// Level j > j0 on block i may start once level j-1 is complete on every row below (i + 1) B + bw, i.e. on the first
// i + lag_dep blocks (lag_dep = ceil(bw / B) + 1): a per-level WATERMARK (number of leading complete blocks) is advanced
// by the warp that completes a block, and waited for with ld.acquire before the gathers.  In the schedule a level
// trails the previous one by lag = lag_dep + slack blocks, the slack covering the tiles the grid has in flight, so that
// a prerequisite was signalled long before it is needed (measured without slack: every step pays the tile latency plus
// the signalling chain, 3x slower than the separate SpMVs).  Prerequisites always lie earlier in
// the sequence and every warp walks the sequence in order, so the earliest unfinished tile can always run: no
// deadlock as long as the grid is co-resident (cooperative launch).  Arithmetic per row is that of spmv_bulk_kernel.
//
// Coherence of the gathers: R_{j+1} is written during the kernel by other SMs and read through L1.  An address is read
// only after its block is complete, L1 is filled per 32-byte sector, and blocks start at multiples of 32 rows of a
// column whose base is 32-byte aligned (setup requires n % 4 == 0), so no sector is ever fetched before it is final:
// L1 never has to be invalidated.  That matters: acquire loads and __threadfence() compile to CCTL.IVALL (drop the SM's
// whole L1), which at one poll / one signal per tile made this kernel 3-5x slower than the separate SpMVs; the kernel
// therefore polls with relaxed loads, signals with a release atomic and fences only when a block completes.
#pragma once
#include "common.cuh"
#include "spmv.cuh"

struct MpkWaveParams {
    int n, nnz, s;
    int j0, nlev;        // levels [j0, j0 + nlev) in this launch
    int tpb;             // tiles (of 32 rows) per block
    int nb;              // blocks
    int lag;             // blocks a level trails the previous one by in the SCHEDULE (dependency distance + slack)
    int lag_dep;         // dependency distance: level j on block i needs level j-1 on the first i + lag_dep blocks
    int basis;
    const int* rp;
    const int* ci;
    const double* va;
    double* R;           // n x s column-major; R(:, j0) is the input
    double* AR;
    const ScgState* st;
    int* done;           // [s][nb] tiles finished per (level, block)   (zeroed before the launch)
    int* watermark;      // [s * 32] leading complete blocks per level, one 128-byte line each (zeroed before the launch)
};

template <int D, int CAP, int WPC>
__global__ void __launch_bounds__(WPC * 32, 3) mpk_wave_kernel(const MpkWaveParams p) {
    if (p.st && p.st->status != SCG_RUNNING) return;
    constexpr int U = 8;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* svals = reinterpret_cast<double*>(smem_raw) + (size_t)warp * D * CAP;
    int* scols = reinterpret_cast<int*>(smem_raw + (size_t)WPC * D * CAP * sizeof(double)) + (size_t)warp * D * CAP;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + (size_t)WPC * D * CAP * 12) + warp * D;
    __shared__ volatile int s_wm[SCG_SMAX];  // the CTA's copy of the watermarks (lower bounds)
    if (threadIdx.x < SCG_SMAX) s_wm[threadIdx.x] = 0;
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < D; d++) mbar_init(&bars[d], 1);
        mbar_fence_init();
    }
    __syncthreads();
    const int n = p.n, nnz = p.nnz, TPB = p.tpb, NB = p.nb;
    // The last nlev - 1 warps of the grid are MANAGERS, one per signalling level: each turns the per-block counters of its
    // level into the level's watermark, so that no worker ever pays for that (a worker that scanned and fenced when it
    // completed a block became the straggler everybody else then waited for: measured 2-4x slower, worse the smaller
    // the blocks).
    const int nman = p.nlev - 1;
    const int GW = (int)gridDim.x * WPC - nman;
    const int gw = (int)blockIdx.x * WPC + warp;
    if (gw >= GW) {
        const int j = p.j0 + (gw - GW);
        int* dj = p.done + (size_t)j * p.nb;
        const int nrt = (p.n + 31) >> 5;
        int w = 0, idle = 0;
        while (w < p.nb) {
            const int w0 = w;
            for (;;) {  // 32 blocks per probe
                const int b = w + lane;
                int ok = 0;
                if (b < p.nb) {
                    int dw;
                    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(dw) : "l"(dj + b) : "memory");
                    ok = dw >= min(p.tpb, nrt - b * p.tpb);
                }
                const unsigned m = __ballot_sync(0xffffffffu, ok);
                const int lead = (m == 0xffffffffu) ? 32 : (__ffs(~m) - 1);
                w += lead;
                if (lead < 32 || w >= p.nb) break;
            }
            if (w > p.nb) w = p.nb;
            if (w > w0) {
                if (lane == 0) {
                    asm volatile("fence.acq_rel.gpu;" ::: "memory");  // the counts (released by the workers) before the publication
                    asm volatile("st.relaxed.gpu.global.s32 [%0], %1;" ::"l"(p.watermark + (size_t)j * 32), "r"(w) : "memory");
                }
                idle = 0;
            } else if (++idle > 4) {
                __nanosleep(200);
            }
            __syncwarp();
        }
        return;
    }
    // TPB is a power of two (setup), so a tile index splits into (q >> LT) = t * nlev + lev and the tile inside the block
    const int LT = 31 - __clz(TPB);
    const unsigned nlevu = (unsigned)p.nlev;
    const unsigned total = (unsigned)(NB + (p.nlev - 1) * p.lag) * nlevu * (unsigned)TPB;  // setup guarantees < 2^31
    const int my_tiles = ((unsigned)gw < total) ? (int)((total - gw + GW - 1) / GW) : 0;
    const int num_row_tiles = (n + 31) >> 5;

    // i-th tile of this warp -> level (relative), block, first row; row0 = -1 for an empty tile
    auto decode = [&](int i, int& lev, int& blk, int& row0) {
        const unsigned q = (unsigned)gw + (unsigned)i * (unsigned)GW;
        const unsigned qq = q >> LT;
        const unsigned t = (nlevu == 2u) ? (qq >> 1) : (nlevu == 4u) ? (qq >> 2) : (nlevu == 3u) ? (__umulhi(qq, 0xAAAAAAABu) >> 1) : qq / nlevu;
        lev = (int)(qq - t * nlevu);
        blk = (int)t - lev * p.lag;
        const int tile = (blk << LT) + (int)(q & (unsigned)(TPB - 1));
        row0 = (blk >= 0 && blk < NB && tile < num_row_tiles) ? tile * 32 : -1;
    };
    auto issue = [&](int i, int nz0, int nz1) {  // as in spmv_bulk_kernel; default L2 policy: the slice is re-read by the next level
        const int sl = i % D;
        const int a0 = nz0 & ~3;
        int bulk_end = (nz1 + 3) & ~3;
        const int lim = nnz & ~3;
        if (bulk_end > lim) bulk_end = lim;
        if (bulk_end < a0) bulk_end = a0;
        const int cnt = bulk_end - a0;
        double* dv = svals + sl * CAP;
        int* dc = scols + sl * CAP;
        if (lane == 0) {
            fence_proxy_async_smem();
            if (cnt > 0) {
                mbar_expect_tx(&bars[sl], (uint32_t)cnt * 12u);
                bulk_g2s_nohint(dv, p.va + a0, (uint32_t)cnt * 8u, &bars[sl]);
                bulk_g2s_nohint(dc, p.ci + a0, (uint32_t)cnt * 4u, &bars[sl]);
            } else {
                mbar_arrive(&bars[sl]);
            }
        }
        const int b_end = __shfl_sync(0xffffffffu, bulk_end, 0);
        const int b_a0 = __shfl_sync(0xffffffffu, a0, 0);
        const int b_nz1 = __shfl_sync(0xffffffffu, nz1, 0);
        for (int e = b_end + lane; e < b_nz1; e += 32) {
            dv[e - b_a0] = p.va[e];
            dc[e - b_a0] = p.ci[e];
        }
    };
    auto tile_bounds = [&](int i, int& nz0, int& nz1) {  // lane 0 only
        int lev, blk, row0;
        decode(i, lev, blk, row0);
        nz0 = nz1 = 0;
        if (row0 >= 0) {
            int row1 = row0 + 32;
            if (row1 > n) row1 = n;
            nz0 = p.rp[row0];
            nz1 = p.rp[row1];
        }
    };

    int nb0 = 0, nb1 = 0;
    for (int i = 0; i < D && i < my_tiles; i++) {
        int a = 0, b = 0;
        if (lane == 0) tile_bounds(i, a, b);
        issue(i, a, b);
    }
    if (lane == 0 && D < my_tiles) tile_bounds(D, nb0, nb1);

    // per-row bounds of the next tile are fetched one step ahead (as in spmv_bulk_kernel); the last watermark seen per
    // level is kept in registers: with the schedule slack most tiles find their prerequisite there and do not poll
    int lev_n, blk_n, row0_n, lo_n = 0, hi_n = 0;
    auto fetch_next = [&](int i) {
        lev_n = 0; blk_n = -1; row0_n = -1; lo_n = hi_n = 0;
        if (i < my_tiles) {
            decode(i, lev_n, blk_n, row0_n);
            const int rown = (row0_n >= 0) ? row0_n + lane : n;
            if (rown < n) { lo_n = p.rp[rown]; hi_n = p.rp[rown + 1]; }
        }
    };
    fetch_next(0);
    // Deferred completion signal.  Counting a tile needs a release (MEMBAR + atomic) that waits for the tile's stores;
    // issued right after the NEXT tile's gathers it waits for nothing the warp would not wait for anyway.  A warp never
    // blocks on a watermark while it holds an unsignalled tile (the poll path signals first), so nobody can wait on it.
    int pend_j = -1, pend_blk = 0;
    auto signal_pending = [&]() {
        if (pend_j >= 0) {
            __syncwarp();  // orders the lanes' stores before lane 0's release (cumulative), as in a grid barrier
            if (lane == 0)
                asm volatile("red.release.gpu.global.add.s32 [%0], 1;" ::"l"(p.done + (size_t)pend_j * NB + pend_blk) : "memory");
            pend_j = -1;
        }
    };
    int wseen[4] = {0, 0, 0, 0};  // watermark of level j0 + l (l < nlev - 1 <= 3 ... larger passes fall back to polling)
    for (int i = 0; i < my_tiles; i++) {
        const int lev = lev_n, blk = blk_n, row0 = row0_n, lo = lo_n, hi = hi_n;
        fetch_next(i + 1);
        const int j = p.j0 + lev;
        const int row = (row0 >= 0) ? row0 + lane : n;
        const bool live = row < n;
        const double* __restrict__ x = p.R + (size_t)j * n;
        // ---- dependency: level j-1 complete on the first blk + lag_dep blocks
        if (lev > 0 && row0 >= 0) {
            int need = blk + p.lag_dep;
            if (need > NB) need = NB;
            int have = 0;
#pragma unroll
            for (int l = 0; l < 4; l++)
                if (l == lev - 1) have = wseen[l];
            if (have < need) {
                signal_pending();
                // next the CTA's shared copy (another warp may have polled since), then global memory with a back-off:
                // thousands of warps polling one address every 64 ns saturate its L2 slice and delay the very
                // publication they wait for (measured: 144 M polls per launch, 55 % of all stall samples)
                int w = 0;
                if (lane == 0) {
                    w = s_wm[lev - 1];
                    unsigned ns = 400;
                    while (w < need) {
                        asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(w) : "l"(p.watermark + (size_t)(j - 1) * 32) : "memory");
                        if (w >= need) break;
                        __nanosleep(ns);
                        if (ns < 3200) ns *= 2;
                    }
                    if (w > s_wm[lev - 1]) s_wm[lev - 1] = w;  // (benign race: any published value is a valid lower bound)
                }
                w = __shfl_sync(0xffffffffu, w, 0);
#pragma unroll
                for (int l = 0; l < 4; l++)
                    if (l == lev - 1) wseen[l] = w;
            }
        }
        // ---- slot -> registers, gathers
        const int sl = i % D;
        const int a0 = __shfl_sync(0xffffffffu, lo, 0) & ~3;
        mbar_wait(&bars[sl], (uint32_t)((i / D) & 1));
        const double* sv = svals + sl * CAP - a0;
        const int* sc = scols + sl * CAP - a0;
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
        signal_pending();  // the previous tile's completion, behind this tile's gathers
        const bool jac = (j + 1 < p.s);
        const int mode = (p.basis == 0) ? 0 : (j == 0 ? 1 : 2);
        double xrow = 0.0, xprev = 0.0;
        if (jac && mode != 0 && live) {
            xrow = x[row];
            if (mode == 2) xprev = p.R[(size_t)(j - 1) * n + row];
        }
        double acc = 0.0;
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
            for (int u = 0; u < U; u++) acc = fma(vv[u], xx[u], acc);
        }
        __syncwarp();  // every lane has read the slot: refill it
        if (i + D < my_tiles) {
            issue(i + D, nb0, nb1);
            if (lane == 0 && i + D + 1 < my_tiles) tile_bounds(i + D + 1, nb0, nb1);
        }
        // same summation order as spmv_bulk_kernel (fragment first, then the remainder)
        double accf = 0.0;
#pragma unroll
        for (int u = 0; u < U; u++) accf = fma(v[u], xv[u], accf);
        acc = accf + acc;
        if (live) {
            p.AR[(size_t)j * n + row] = acc;
            if (jac) {
                double z = __drcp_rn(diag) * acc;
                if (mode == 1) z = z - xrow;
                else if (mode == 2) z = 2.0 * (z - xrow) - xprev;
                p.R[(size_t)(j + 1) * n + row] = z;
            }
        }
        // ---- completion is signalled one tile late (see signal_pending): remember this tile
        if (row0 >= 0 && lev + 1 < p.nlev) { pend_j = j; pend_blk = blk; }
    }
    signal_pending();
}

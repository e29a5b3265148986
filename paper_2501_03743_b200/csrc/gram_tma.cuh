// gram_tma.cuh -- steps a2 + a3 for s >= 5: the same fused block inner products as gram.cuh (same entries, same
// deterministic cross-block finish and on-device solves), but the operands are streamed through shared memory by a
// producer warp with the TMA engine (tile_pipe.cuh), so that ~200 KB per SM are in flight independent of the
// registers the accumulators take.
//
// CTA = NWC consumer warps + NPW producer warps, one persistent CTA per SM.
// Tile = T rows; slot = { R[S][T+2] | AR[S][T+2] | AP[T*S+2] | r[T+2] } doubles; ring of D slots.
// Consumer lanes: NSL lanes share one row, lane slice q owns the G columns q*G .. q*G+G-1 of AR / AP:
//   accM[i][g] += R_i * AR_{qG+g}     accC[g][j] += AP_{qG+g} * R_j     accm[g] += R_{qG+g} * r
// lane = rlo + 2*q + 2*NSL*rhi, row inside the pass = rlo + 2*rhi.  With this order the 8 lanes of a 128-bit
// shared-memory phase read 8 different 16-byte chunks of two consecutive interleaved AP rows (s = 8: bank-conflict
// free), and a column read touches 32/NSL consecutive doubles (one wavefront, broadcast to the NSL lanes of a row).
#pragma once
#include "gram.cuh"
#include "tile_pipe.cuh"

template <int S>
struct GramTmaCfg {
    static constexpr int NSL = (S <= 4) ? 1 : (S <= 6) ? 2 : (S <= 8) ? 4 : 8;   // lanes (slices) per row
    static constexpr int G = (S + NSL - 1) / NSL;                                // columns per slice
    static constexpr int NACC = 2 * S * G + G;
    static constexpr int RPP = 32 / NSL;                                         // rows per warp pass
    static constexpr int NWC = 8;                                                // consumer warps
    static constexpr int T = (S <= 4) ? 512 : (S == 5) ? 384 : (S <= 8) ? 128 : 64;   // rows per tile (s <= 5: few large copies in flight)
    static constexpr int PASSES = T / (NWC * RPP);
    static constexpr int COLS = T + 2;                                           // column slice + alignment slack
    static constexpr int OFF_AR = S * COLS, OFF_AP = 2 * S * COLS, OFF_r = OFF_AP + T * S + 2;
    static constexpr int SLOT = OFF_r + COLS;                     // doubles per slot (every sub-buffer 16 B aligned)
    static constexpr int D_FIT = ((S <= 8 ? 192 : 144) * 1024) / (SLOT * 8);  // one CTA per SM: the ring takes most of its shared memory
    static constexpr int D = D_FIT > 8 ? 8 : (D_FIT < 2 ? 2 : D_FIT);
    static constexpr int NSEG = 2 * S + 2;
    static constexpr int NPW = (S <= 5) ? 3 : 4;                  // producer warps (tile i is filled by warp i % NPW)
    static constexpr int THREADS = (NWC + NPW) * 32;
    static constexpr size_t SMEM = (size_t)D * SLOT * sizeof(double) + 2 * D * sizeof(uint64_t);
    static_assert(PASSES >= 1 && T % (NWC * RPP) == 0, "tile must hold whole passes of all consumer warps");
    static_assert(NPW <= D, "a producer may run at most one phase ahead of a slot (parity wait): needs NPW <= D");
};

// sum over the lanes that share a slice: lane bit 0 (rlo) and the bits above the slice field (rhi)
template <int NSL>
__device__ __forceinline__ double slice_sum(double v) {
    v += __shfl_xor_sync(0xffffffffu, v, 1);
#pragma unroll
    for (int o = 2 * NSL; o < 32; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <int S>
__global__ void __launch_bounds__(GramTmaCfg<S>::THREADS, 1)
gram_tma_kernel(int64_t n, const double* __restrict__ R, const double* __restrict__ AR, const double* __restrict__ AP,
                const double* __restrict__ r, double* __restrict__ partials, ScgState* __restrict__ st, int do_solve,
                int64_t num_tiles) {
    using TC = GramTmaCfg<S>;
    constexpr int G = TC::G, NSL = TC::NSL, NWC = TC::NWC, NACC = TC::NACC, RPP = TC::RPP;
    constexpr int T = TC::T, COLS = TC::COLS, D = TC::D;
    pdl_wait();  // (common.cuh: the predecessor in the graph may still be draining)
    pdl_launch();
    if (st->status != SCG_RUNNING) return;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* slots = reinterpret_cast<double*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)D * TC::SLOT * sizeof(double));
    uint64_t* empty = full + D;
    __shared__ double red[NWC * NSL][NACC];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int d = 0; d < D; d++) { mbar_init(&full[d], 1); mbar_init(&empty[d], NWC); }
        mbar_fence_init();
    }
    __syncthreads();
    const int64_t my_tiles = ((int64_t)blockIdx.x < num_tiles) ? (num_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;

    if (warp >= NWC) {
        // ------------------------------------------------ producer warps (one warp sustains only ~15 GB/s of bulk copies)
        const uint64_t policy = l2_policy_evict_first();
        const int64_t ns = (int64_t)S * n;
        for (int64_t i = warp - NWC; i < my_tiles; i += TC::NPW) {
            const int sl = (int)(i % D);
            if (i >= D) mbar_wait(&empty[sl], (uint32_t)(((i / D) - 1) & 1));
            const int64_t row0 = ((int64_t)blockIdx.x + i * gridDim.x) * T;
            const int cnt = (int)((n - row0 < T) ? (n - row0) : T);
            double* sb = slots + (size_t)sl * TC::SLOT;
            auto make_seg = [&](int c) {
                TileSeg sg;
                sg.cnt = cnt;
                if (c < S) { sg.g = R + (int64_t)c * n + row0; sg.buf_end = R + ns; sg.dst = sb + c * COLS; }
                else if (c < 2 * S) { sg.g = AR + (int64_t)(c - S) * n + row0; sg.buf_end = AR + ns; sg.dst = sb + TC::OFF_AR + (c - S) * COLS; }
                else if (c == 2 * S) { sg.g = AP + row0 * S; sg.buf_end = AP + ns; sg.dst = sb + TC::OFF_AP; sg.cnt = cnt * S; }
                else { sg.g = r + row0; sg.buf_end = r + n; sg.dst = sb + TC::OFF_r; }
                return sg;
            };
            tile_fill(TC::NSEG, make_seg, &full[sl], policy, lane);
        }
    } else {
        // ------------------------------------------------ consumer warps
        const int q = (lane >> 1) & (NSL - 1), c0 = q * G;
        const int rip = (lane & 1) + 2 * (lane / (2 * NSL));  // row inside the pass
        double accM[S][G], accC[G][S], accm[G];
#pragma unroll
        for (int g = 0; g < G; g++) {
            accm[g] = 0.0;
#pragma unroll
            for (int i = 0; i < S; i++) { accM[i][g] = 0.0; accC[g][i] = 0.0; }
        }
        for (int64_t i = 0; i < my_tiles; i++) {
            const int sl = (int)(i % D);
            const int64_t row0 = ((int64_t)blockIdx.x + i * gridDim.x) * T;
            const int cnt = (int)((n - row0 < T) ? (n - row0) : T);
            const double* sb = slots + (size_t)sl * TC::SLOT;
            // leading doubles to skip in the column sub-buffers (copies start at 16-byte aligned addresses); the
            // interleaved AP tile starts aligned (base 16-byte aligned, row0 * S even)
            int shR[S], shAR[G];
#pragma unroll
            for (int j = 0; j < S; j++) shR[j] = seg_shift(R + (int64_t)j * n + row0);
#pragma unroll
            for (int g = 0; g < G; g++) shAR[g] = seg_shift(AR + (int64_t)((c0 + g < S) ? c0 + g : 0) * n + row0);
            const int shr = seg_shift(r + row0);
            mbar_wait(&full[sl], (uint32_t)((i / D) & 1));
#pragma unroll
            for (int p = 0; p < TC::PASSES; p++) {
                const int lr = (p * NWC + warp) * RPP + rip;  // row inside the tile
                if (lr < cnt) {
                    double Rv[S], ARv[G], APv[G], Rsel[G];
#pragma unroll
                    for (int j = 0; j < S; j++) Rv[j] = sb[j * COLS + shR[j] + lr];
                    if constexpr (G == 2 && S % 2 == 0) {
                        const double2 a2 = *reinterpret_cast<const double2*>(sb + TC::OFF_AP + lr * S + c0);
                        APv[0] = a2.x;
                        APv[1] = a2.y;
                    } else {
#pragma unroll
                        for (int g = 0; g < G; g++) APv[g] = (c0 + g < S) ? sb[TC::OFF_AP + lr * S + c0 + g] : 0.0;
                    }
#pragma unroll
                    for (int g = 0; g < G; g++) {
                        const bool ok = (G * NSL == S) || (c0 + g < S);
                        const int c = ok ? c0 + g : 0;
                        const double a = sb[TC::OFF_AR + c * COLS + shAR[g] + lr];
                        ARv[g] = ok ? a : 0.0;
                        if constexpr (NSL == 1) Rsel[g] = Rv[g];
                        else {
                            const double d = sb[c * COLS + seg_shift(R + (int64_t)c * n + row0) + lr];
                            Rsel[g] = ok ? d : 0.0;
                        }
                        if (!ok) APv[g] = 0.0;
                    }
                    const double rv = sb[TC::OFF_r + shr + lr];
#pragma unroll
                    for (int g = 0; g < G; g++) {
#pragma unroll
                        for (int i2 = 0; i2 < S; i2++) {
                            accM[i2][g] = fma(Rv[i2], ARv[g], accM[i2][g]);
                            accC[g][i2] = fma(APv[g], Rv[i2], accC[g][i2]);
                        }
                        accm[g] = fma(Rsel[g], rv, accm[g]);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[sl]);
        }
        // ---- in-warp reduction over the lanes of each slice; lane 2q holds slice q ----
        const bool writer = (lane & 1) == 0 && (lane / (2 * NSL)) == 0;
#pragma unroll
        for (int g = 0; g < G; g++) {
#pragma unroll
            for (int i = 0; i < S; i++) {
                const double a = slice_sum<NSL>(accM[i][g]);
                const double b = slice_sum<NSL>(accC[g][i]);
                if (writer) { red[warp * NSL + q][i * G + g] = a; red[warp * NSL + q][S * G + g * S + i] = b; }
            }
            const double c = slice_sum<NSL>(accm[g]);
            if (writer) red[warp * NSL + q][2 * S * G + g] = c;
        }
    }
    gram_cross_block_finish<S, G, NSL, NWC>(red, partials, st, do_solve);
}

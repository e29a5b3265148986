// update_tma.cuh -- step a4 (+ a5) for s >= 5: the same fused block update as update.cuh (same arithmetic per row,
// same deterministic ||r||^2 finish and stop test), with every operand streamed through shared memory by a producer
// warp and the TMA engine (tile_pipe.cuh).  One consumer thread per row of the tile; the new P / AP rows return
// through the slot and leave as bulk stores (one contiguous segment per warp); x, r, R_1 are coalesced stores.
//
// Slot = { R[S][T+2] | AR[S][T+2] | P[T*S+2] | AP[T*S+2] | x[T+2] | r[T+2] | dinv[T+2] } doubles; ring of D slots.
#pragma once
#include "tile_pipe.cuh"
#include "update.cuh"

template <int S>
struct UpdateTmaCfg {
    static constexpr int T = (S <= 4) ? 256 : (S <= 8) ? 128 : 64;
    static constexpr int NCW = T / 32;                           // consumer warps
    static constexpr int COLS = T + 2;
    static constexpr int OFF_AR = S * COLS, OFF_P = 2 * S * COLS, OFF_AP = OFF_P + T * S + 2, OFF_x = OFF_AP + T * S + 2,
                         OFF_r = OFF_x + COLS, OFF_d = OFF_r + COLS;
    static constexpr int SLOT = OFF_d + COLS;
    static constexpr int D = 3;
    static constexpr int NSEG = 2 * S + 5;
    static constexpr int NPW = 3;                                // producer warps (tile i is filled by warp i % NPW)
    static constexpr int THREADS = (NCW + NPW) * 32;
    static constexpr int MINB = (S <= 8) ? 2 : 1;
    static constexpr size_t SMEM = (size_t)D * SLOT * sizeof(double) + 2 * D * sizeof(uint64_t);
    static_assert(NPW <= D, "a producer may run at most one phase ahead of a slot (parity wait): needs NPW <= D");
};

// one interleaved row (S doubles) from shared memory; 128-bit loads when S is even (the tile starts 16-byte aligned)
template <int S>
__device__ __forceinline__ void load_row(const double* __restrict__ src, double (&v)[S]) {
    if constexpr (S % 2 == 0) {
        const double2* s2 = reinterpret_cast<const double2*>(src);
#pragma unroll
        for (int l = 0; l < S / 2; l++) { const double2 a = s2[l]; v[2 * l] = a.x; v[2 * l + 1] = a.y; }
    } else {
#pragma unroll
        for (int l = 0; l < S; l++) v[l] = src[l];
    }
}

template <int S, bool MOM>
__global__ void __launch_bounds__(UpdateTmaCfg<S>::THREADS, UpdateTmaCfg<S>::MINB)
update_tma_kernel(int64_t n, double* __restrict__ R, const double* __restrict__ AR, double* __restrict__ P,
                  double* __restrict__ AP, double* __restrict__ x, double* __restrict__ r, const double* __restrict__ dinv,
                  const double* __restrict__ beta_g, const double* __restrict__ alpha_g, double* __restrict__ partials,
                  ScgState* __restrict__ st, double* __restrict__ rho_out, int64_t num_tiles) {
    using TC = UpdateTmaCfg<S>;
    constexpr int T = TC::T, COLS = TC::COLS, D = TC::D, NCW = TC::NCW;
    pdl_wait();  // (common.cuh: the predecessor in the graph may still be draining)
    pdl_launch();
    if (st->status != SCG_RUNNING) return;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* slots = reinterpret_cast<double*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)D * TC::SLOT * sizeof(double));
    uint64_t* empty = full + D;
    __shared__ __align__(16) double sbeta[S * S];
    __shared__ double salpha[S];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int e = threadIdx.x; e < S * S; e += blockDim.x) sbeta[e] = beta_g[e];
    if (threadIdx.x < S) salpha[threadIdx.x] = alpha_g[threadIdx.x];
    if (threadIdx.x == 0) {
#pragma unroll
        for (int d = 0; d < D; d++) { mbar_init(&full[d], 1); mbar_init(&empty[d], NCW); }
        mbar_fence_init();
    }
    __syncthreads();

    double rho = 0.0, mu0 = 0.0;
    const int64_t my_tiles = ((int64_t)blockIdx.x < num_tiles) ? (num_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;

    if (warp >= NCW) {
        // ------------------------------------------------ producer warps
        const uint64_t policy = l2_policy_evict_first();
        const int64_t ns = (int64_t)S * n;
        for (int64_t i = warp - NCW; i < my_tiles; i += TC::NPW) {
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
                else if (c == 2 * S) { sg.g = P + row0 * S; sg.buf_end = P + ns; sg.dst = sb + TC::OFF_P; sg.cnt = cnt * S; }
                else if (c == 2 * S + 1) { sg.g = AP + row0 * S; sg.buf_end = AP + ns; sg.dst = sb + TC::OFF_AP; sg.cnt = cnt * S; }
                else if (c == 2 * S + 2) { sg.g = x + row0; sg.buf_end = x + n; sg.dst = sb + TC::OFF_x; }
                else if (c == 2 * S + 3) { sg.g = r + row0; sg.buf_end = r + n; sg.dst = sb + TC::OFF_r; }
                else { sg.g = dinv + row0; sg.buf_end = dinv + n; sg.dst = sb + TC::OFF_d; }
                return sg;
            };
            tile_fill(TC::NSEG, make_seg, &full[sl], policy, lane);
        }
    } else {
        // ------------------------------------------------ consumer warps: one thread per row of the tile
        const int lr = warp * 32 + lane;
        for (int64_t i = 0; i < my_tiles; i++) {
            const int sl = (int)(i % D);
            const int64_t row0 = ((int64_t)blockIdx.x + i * gridDim.x) * T;
            const int cnt = (int)((n - row0 < T) ? (n - row0) : T);
            double* sb = slots + (size_t)sl * TC::SLOT;
            const bool live = lr < cnt;
            const int64_t row = row0 + lr;
            double vP[S], oP[S], vA[S], oA[S];
            double x0 = 0.0, r0 = 0.0, di = 0.0;
            mbar_wait(&full[sl], (uint32_t)((i / D) & 1));
            if (live) {
                // P / AP bases are 16-byte aligned (checked at dispatch) and row0 * S is even: the tiles start at shift 0
                load_row<S>(sb + TC::OFF_P + lr * S, vP);
                load_row<S>(sb + TC::OFF_AP + lr * S, vA);
#pragma unroll
                for (int j = 0; j < S; j++) {
                    oP[j] = sb[j * COLS + seg_shift(R + (int64_t)j * n + row0) + lr];
                    oA[j] = sb[TC::OFF_AR + j * COLS + seg_shift(AR + (int64_t)j * n + row0) + lr];
                }
                x0 = sb[TC::OFF_x + seg_shift(x + row0) + lr];
                r0 = sb[TC::OFF_r + seg_shift(r + row0) + lr];
                di = sb[TC::OFF_d + seg_shift(dinv + row0) + lr];
            }
            double xi = 0.0, ri = 0.0;
            if (live) {
                xi = update_row<S>(vP, oP, sbeta, salpha, x0, 1.0);    // P <- R + P beta ; x += P alpha
                ri = update_row<S>(vA, oA, sbeta, salpha, r0, -1.0);   // AP <- AR + AP beta ; r -= AP alpha
            }
            if constexpr (S % 2 == 0) {
                // new P / AP rows go back into the slot (each thread over the row it read) and leave as two bulk
                // stores per warp: 32 rows = one contiguous, fully coalesced segment of the interleaved block
                if (live) {
                    store_row<S>(sb + TC::OFF_P + lr * S, oP);
                    store_row<S>(sb + TC::OFF_AP + lr * S, oA);
                }
                fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) {
                    const int rows_w = cnt - warp * 32 < 32 ? cnt - warp * 32 : 32;
                    if (rows_w > 0) {
                        const uint32_t bytes = (uint32_t)rows_w * S * 8u;
                        bulk_s2g(P + (row0 + warp * 32) * S, sb + TC::OFF_P + warp * 32 * S, bytes);
                        bulk_s2g(AP + (row0 + warp * 32) * S, sb + TC::OFF_AP + warp * 32 * S, bytes);
                        bulk_commit();
                    }
                }
            } else {
                if (live) {
                    store_row<S>(P + row * S, oP);
                    store_row<S>(AP + row * S, oA);
                }
            }
            if (live) {
                x[row] = xi;
                r[row] = ri;
                const double r1 = di * ri;
                R[row] = r1;  // R(:,1) of the next outer iteration
                rho = fma(ri, ri, rho);
                if (MOM) mu0 = fma(r1, ri, mu0);
            }
            if (lane == 0) {
                if constexpr (S % 2 == 0) bulk_wait_read();  // the stores have read the slot: it may be refilled
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[sl]);
        }
        if (lane == 0) bulk_wait_all();
    }
    update_block_finish<MOM>(rho, mu0, NCW, partials, st, rho_out);
}

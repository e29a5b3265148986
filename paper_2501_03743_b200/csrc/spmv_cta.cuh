// spmv_cta.cuh -- step a1 for stencil-like matrices (one lane per row: mean row <= 8 entries, every 7-point config; two lanes
// per row: mean rows of 16-32 entries, the 27-point config): the Jacobi-fused CSR SpMV of the matrix-powers kernel
// (Alg. 4) with a CTA-wide producer / consumer TMA pipeline.
//
// Why a second bulk-staged kernel (round 2).  The per-warp rings of spmv_bulk_kernel keep 24 warps x 2 slots x 2 arrays
// = 96 bulk copies of ~1.3 KB in flight per SM.  Measured on this B200 with a pure streaming kernel
// (sstep_cg_measure_bandwidth variants 2-5, measure.cuh; numbers in DESIGN.md section 6): the 1-D bulk-copy path of an SM runs at full speed only up to ~32 copies in flight --
// 16-32 copies of >= 4 KB stream 7.2-7.3 TB/s from HBM and 18 TB/s from L2, 48 copies 6.0-7.5 TB/s from either, 96
// copies 3.6 TB/s.  So the bytes in flight must come from FEW, LARGE copies: here one producer warp per CTA streams
// tiles of TR = 256 rows (colidx + vals of the whole tile = two copies of ~14 KB + ~7 KB) into a ring of D stages, and
// TR/32 consumer warps compute from shared memory: 3 CTAs x D = 3 stages x 2 = 18 copies and ~190 KB in flight per SM.
//
//   producer (warp TR/32):  wait empty[st] -> rowptr of the tile's ends -> expect_tx(full[st]) + 2 bulk copies
//   consumer warp w:        rows tile*TR + 32 w + lane; (rowptr pair fetched one tile ahead) wait full[st] -> fragment
//                           (<= 8 entries) to registers -> x gathers issued -> arrive empty[st] -> FMAs, epilogue, stores
// Arithmetic per row, epilogue modes, 1/a_ii from the row's own diagonal entry and the moment partials (MOM) are those
// of spmv_bulk_kernel at L = 1 (spmv.cuh), bit for bit.  Tiles are dealt to CTAs round-robin, so the grid sweeps one
// contiguous window of rows (gather locality in L1 / L2).
#pragma once
#include "common.cuh"
#include "spmv.cuh"

// One row per lane out of a staged tile: acc = sum_k a_k x[col_k] over the row's entries [lo, hi) (sv / sc = the stage's
// vals / cols, pre-offset so that they are indexed by the global nnz index), the fragment of <= 8 entries summed in
// ascending order, then the remainder of longer rows -- the order of spmv_bulk_kernel at L = 1, bit for bit.
// Lean on purpose (the SpMV issues ~230 instructions per 32 rows and runs at ~50 % issue utilisation, which is what
// bounds a level served from L2): entries past the row's end re-read the row's FIRST entry with the value masked to
// zero, so that the index and the gather need no predicate (the gathered column is a genuine neighbour of this row,
// hence a valid index whose x cannot be non-finite unless the row's true result already is); `lo` must be a staged
// index also for empty / dead rows.  Two phases, so that the caller can hand the stage back between them.  UNI: the diagonal is constant (every Poisson config), 1 / a_ii is a kernel argument
// and the pick-up of a_ii from the row disappears; else diag returns the row's own diagonal entry.
template <int U>
struct StageRowFrag {
    double v[U], xv[U];
    double rem, diag;
};
// phase 1: fragment to registers, gathers issued (after it the stage may be handed back).  L lanes share a row: lane g of
// the group takes the entries lo + g, lo + g + L, ...; U per lane live in registers, longer rows go through the remainder.
template <bool UNI, int L, int U>
__device__ __forceinline__ void stage_row_load(const double* sv, const int* sc, int lo, int hi, int row, int g,
                                               const double* __restrict__ x, StageRowFrag<U>& f) {
    int c[U];
    f.diag = 0.0;
#pragma unroll
    for (int u = 0; u < U; u++) {
        const int kk = lo + g + u * L;
        const bool ok = kk < hi;
        const int k2 = ok ? kk : lo;
        c[u] = sc[k2];
        const double t = sv[k2];
        f.v[u] = ok ? t : 0.0;
        if (!UNI) { if (ok && c[u] == row) f.diag = t; }
    }
#pragma unroll
    for (int u = 0; u < U; u++) f.xv[u] = x[c[u]];
    double rem = 0.0;
    for (int k0 = lo + g + U * L; k0 < hi; k0 += 8 * L) {  // rows longer than U L entries: further batches of 8 per lane
        int cc[8];
        double vv[8], xx[8];
#pragma unroll
        for (int u = 0; u < 8; u++) {
            const int kk = k0 + u * L;
            const bool ok = kk < hi;
            cc[u] = ok ? sc[kk] : -1;
            vv[u] = ok ? sv[kk] : 0.0;
            if (!UNI) { if (cc[u] == row) f.diag = vv[u]; }
        }
#pragma unroll
        for (int u = 0; u < 8; u++) xx[u] = (cc[u] >= 0) ? x[cc[u]] : 0.0;
#pragma unroll
        for (int u = 0; u < 8; u++) rem = fma(vv[u], xx[u], rem);
    }
    f.rem = rem;
}
// phase 2: the lane's partial row sum (waits for the gathers); the caller adds the L lanes of a row with group_sum<L>
template <int U>
__device__ __forceinline__ double stage_row_sum(const StageRowFrag<U>& f) {
    double acc = 0.0;
#pragma unroll
    for (int u = 0; u < U; u++) acc = fma(f.v[u], f.xv[u], acc);
    return acc + f.rem;
}

template <int D, int TR, int CAPT, int L>
struct SpmvCtaCfg {
    static constexpr int NCW = TR * L / 32;                  // consumer warps (a warp covers 32 / L rows)
    static constexpr int THREADS = NCW * 32 + 32;            // + one producer warp
    static constexpr size_t STAGE = (size_t)CAPT * 12;       // vals then cols of one stage
    static constexpr size_t SMEM = (size_t)D * STAGE + (size_t)D * 16 /* full, empty */ + (size_t)D * 8 /* a0 per stage */;
    static_assert(CAPT % 4 == 0 && (TR * L) % 32 == 0, "stage sub-buffers must stay 16-byte aligned");
};

template <int D, int TR, int CAPT, bool MOM, int MINB, bool UNI, int L = 1, int U = 8>
__global__ void __launch_bounds__(TR * L + 32, MINB)
spmv_cta_kernel(int n, int nnz, const int* __restrict__ rp, const int* __restrict__ ci, const double* __restrict__ va,
                const double* __restrict__ x, double* __restrict__ y, double* __restrict__ yjac,
                const double* __restrict__ xprev, int mode, const ScgState* __restrict__ st, int num_tiles,
                double* __restrict__ mom_a, double* __restrict__ mom_b, double dinv_uniform) {
    using Cfg = SpmvCtaCfg<D, TR, CAPT, L>;
    constexpr int NCW = Cfg::NCW, RPW = 32 / L;  // rows per consumer warp
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* svals = reinterpret_cast<double*>(smem_raw);                                  // [D][CAPT]
    int* scols = reinterpret_cast<int*>(smem_raw + (size_t)D * CAPT * sizeof(double));    // [D][CAPT]
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)D * Cfg::STAGE);
    uint64_t* empty = full + D;
    int* s_a0 = reinterpret_cast<int*>(empty + D);                                        // [D] first staged nnz index
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
#pragma unroll
        for (int d = 0; d < D; d++) { mbar_init(&full[d], 1); mbar_init(&empty[d], NCW); }
        mbar_fence_init();
    }
    __syncthreads();
    const int my_tiles = ((int)blockIdx.x < num_tiles) ? (num_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    auto tile_row0 = [&](int i) { return ((int)blockIdx.x + i * (int)gridDim.x) * TR; };

    if (warp == NCW) {
        // ------------------------------------------------------------------ producer warp
        // rowptr / colidx / vals are written by no kernel: the first D tiles are staged ahead of the dependency wait (with
        // a programmatic dependent launch they stream while the predecessor drains); if the solver has stopped, producer
        // and consumers agree to handle exactly those D tiles (the consumers only hand them back)
        const uint64_t policy = l2_policy_evict_first();
        int tiles_eff = my_tiles;
        for (int i = 0; i < tiles_eff; i++) {
            const int sl = i % D;
            if (i == D) {  // ring filled once: from here on the solver's state decides (a stopped solver streams no further)
                pdl_wait();
                if (st && st->status != SCG_RUNNING) break;
            }
            if (i >= D) mbar_wait(&empty[sl], (uint32_t)(((i / D) - 1) & 1));
            const int row0 = tile_row0(i);
            int row1 = row0 + TR;
            if (row1 > n) row1 = n;
            int nz0 = 0, nz1 = 0;
            if (lane == 0) { nz0 = rp[row0]; nz1 = rp[row1]; }
            nz0 = __shfl_sync(0xffffffffu, nz0, 0);
            nz1 = __shfl_sync(0xffffffffu, nz1, 0);
            const int a0 = nz0 & ~3;
            int bulk_end = (nz1 + 3) & ~3;
            const int lim = nnz & ~3;
            if (bulk_end > lim) bulk_end = lim;
            if (bulk_end < a0) bulk_end = a0;
            const int cnt = bulk_end - a0;
            double* dv = svals + (size_t)sl * CAPT;
            int* dc = scols + (size_t)sl * CAPT;
            // ragged tail of the arrays (at most 3 entries of the whole matrix) by plain loads
            for (int e = bulk_end + lane; e < nz1; e += 32) { dv[e - a0] = va[e]; dc[e - a0] = ci[e]; }
            if (lane == 0) s_a0[sl] = a0;
            __syncwarp();  // the stores above are ordered before lane 0's releasing arrive
            if (lane == 0) {
                fence_proxy_async_smem();
                if (cnt > 0) {
                    mbar_expect_tx(&full[sl], (uint32_t)cnt * 12u);
                    bulk_g2s(dv, va + a0, (uint32_t)cnt * 8u, &full[sl], policy);
                    bulk_g2s(dc, ci + a0, (uint32_t)cnt * 4u, &full[sl], policy);
                } else {
                    mbar_arrive(&full[sl]);
                }
            }
        }
        if (MOM) spmv_moment_finish(0.0, 0.0, mom_a, mom_b);  // (block-wide reduction: every warp takes part)
        return;
    }

    // ---------------------------------------------------------------------- consumer warps
    double ma = 0.0, mb = 0.0;
    const bool jac = yjac != nullptr;
    int lo_n = 0, hi_n = 0;
    auto row_bounds = [&](int i, int& lo, int& hi) {
        lo = hi = 0;
        if (i < my_tiles) {
            const int row = tile_row0(i) + warp * RPW + lane / L;
            if (row < n) { lo = rp[row]; hi = rp[row + 1]; }
        }
    };
    row_bounds(0, lo_n, hi_n);  // (rowptr only: may run ahead of the dependency wait)
    pdl_wait();
    pdl_launch();
    const bool running = !(st && st->status != SCG_RUNNING);
    const int tiles_eff = running ? my_tiles : (my_tiles < D ? my_tiles : D);  // stopped: only what the prologue staged
    for (int i = 0; i < tiles_eff; i++) {
        const int sl = i % D;
        const int lo = lo_n, hi = hi_n;
        const int row = tile_row0(i) + warp * RPW + lane / L;
        const int g = lane % L;
        row_bounds(i + 1, lo_n, hi_n);
        mbar_wait(&full[sl], (uint32_t)((i / D) & 1));
        if (!running) {  // stopped solver: hand the stage back, compute nothing
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[sl]);
            continue;
        }
        const int a0 = s_a0[sl];
        const double* sv = svals + (size_t)sl * CAPT - a0;
        const int* sc = scols + (size_t)sl * CAPT - a0;
        const bool live = row < n;
        StageRowFrag<U> f;
        stage_row_load<UNI, L, U>(sv, sc, live ? lo : a0, live ? hi : a0, row, g, x, f);
        double xrow = 0.0, xpv = 0.0;
        if ((MOM || (jac && mode != 0)) && live && g == 0) {
            xrow = x[row];
            if (mode == 2) xpv = xprev[row];
        }
        __syncwarp();  // every lane has read the stage
        if (lane == 0) mbar_arrive(&empty[sl]);
        const double acc = group_sum<L>(stage_row_sum<U>(f));
        double diag = f.diag;
        if (L > 1 && !UNI && jac) diag = group_sum<L>(diag);  // exactly one lane of the group holds a_ii, the others 0
        if (live && g == 0) {
            y[row] = acc;
            if (MOM) ma = fma(xrow, acc, ma);
            if (jac) {
                double z = (UNI ? dinv_uniform : __drcp_rn(diag)) * acc;
                if (MOM) mb = fma(z, acc, mb);
                if (mode == 1) z = z - xrow;
                else if (mode == 2) z = 2.0 * (z - xrow) - xpv;
                yjac[row] = z;
            }
        }
    }
    if (MOM) spmv_moment_finish(ma, mb, mom_a, mom_b);
}

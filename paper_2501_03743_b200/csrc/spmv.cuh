// spmv.cuh -- step a1 of the hot path: one Jacobi-fused CSR SpMV of the matrix-powers kernel
// (Alg. 4):  y = A x  (AR_j = A R_j)  and, in the epilogue,
//   mode 0 (monomial):        yjac = dinv .* y                      (R_{j+1} = B^-1 AR_j)
//   mode 1 (Chebyshev, j=1):  yjac = dinv .* y - x                  (R_2 = Z R_1,  Z = D^-1 A - I)
//   mode 2 (Chebyshev, j>1):  yjac = 2 (dinv .* y - x) - xprev      (R_{j+1} = 2 Z R_j - R_{j-1})
// Two variants, chosen at setup from the row-length statistics:
//   spmv_vec_kernel  : generic vector-per-row (L lanes per row, L in {1..32}); any CSR.
//   spmv_bulk_kernel : per-warp multi-stage pipeline; the warp's slice of colidx/vals is streamed into
//                      shared memory by the TMA engine (cp.async.bulk, 16 B aligned, L2 evict-first) while the
//                      warp gathers x for the previous tile.  Needs every tile of 32/L rows to hold < CAP-3 nnz.
// 1/a_ii: the bulk kernel takes it from the row's own diagonal entry (__drcp_rn = the IEEE quotient 1/a_ii, the same
// bits as the dinv array the generic kernel reads).
#pragma once
#include "common.cuh"

__device__ __forceinline__ void spmv_epilogue(int64_t row, double acc, const double* __restrict__ dinv,
                                              const double* __restrict__ x, const double* __restrict__ xprev, int mode,
                                              double* __restrict__ y, double* __restrict__ yjac) {
    y[row] = acc;
    if (yjac) {
        double z = dinv[row] * acc;
        if (mode == 1) z = z - x[row];
        else if (mode == 2) z = 2.0 * (z - x[row]) - xprev[row];
        yjac[row] = z;
    }
}

// Moment form: per-block partial sums of  mu_a = sum_rows x_i (A x)_i  and  mu_b = sum_rows (D^-1 A x)_i (A x)_i
// (for SpMV j of the MPK these are mu^{2j-1} = R_j^T AR_j and mu^{2j} = R_{j+1}^T AR_j; Eq. 4).
// Every thread of the CTA calls; one double per block and moment, summed later in fixed block order by sw_kernel.
__device__ __forceinline__ void spmv_moment_finish(double ma, double mb, double* __restrict__ mom_a, double* __restrict__ mom_b) {
    __shared__ double red[2][32];
    ma = warp_sum(ma);
    mb = warp_sum(mb);
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = ma; red[1][threadIdx.x >> 5] = mb; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) { a += red[0][w]; b += red[1][w]; }
        mom_a[blockIdx.x] = a;
        if (mom_b) mom_b[blockIdx.x] = b;
    }
}

template <int L, bool MOM>
__global__ void __launch_bounds__(256) spmv_vec_kernel(int64_t n, const int* __restrict__ rp, const int* __restrict__ ci,
                                                       const double* __restrict__ va, const double* __restrict__ dinv,
                                                       const double* __restrict__ x, double* __restrict__ y,
                                                       double* __restrict__ yjac, const double* __restrict__ xprev, int mode,
                                                       const ScgState* __restrict__ st, double* __restrict__ mom_a,
                                                       double* __restrict__ mom_b) {
    pdl_wait();
    pdl_launch();
    if (st && st->status != SCG_RUNNING) return;
    double ma = 0.0, mb = 0.0;  // moment partials x^T (A x) and (D^-1 A x)^T (A x), see spmv_moment_finish
    const int g = threadIdx.x % L;
    const int64_t rows_per_pass = (int64_t)gridDim.x * (blockDim.x / L);
    // the loop runs on the warp's first row so that all 32 lanes reach the shuffles the same number of times
    const int warp_rows = 32 / L;
    for (int64_t wrow = (int64_t)blockIdx.x * (blockDim.x / L) + (threadIdx.x >> 5) * warp_rows; wrow < n;
         wrow += rows_per_pass) {
        const int64_t row = wrow + (threadIdx.x & 31) / L;
        const bool live = row < n;
        int lo = 0, hi = 0;
        if (live) { lo = rp[row]; hi = rp[row + 1]; }
        double acc = 0.0;
        // plain loop on purpose: batching the index/value loads by hand measured the same (27-point 160^3: 273.7 vs
        // 272.7 us -- the kernel sits at ~70 % of the L1 wavefront rate, not on latency) and streaming hints on them
        // 20-90 % slower -- consecutive iterations re-use the sectors of colidx/vals through L1
        for (int k = lo + g; k < hi; k += L) acc = fma(va[k], x[ci[k]], acc);
        acc = group_sum<L>(acc);
        if (live && g == 0) {
            spmv_epilogue(row, acc, dinv, x, xprev, mode, y, yjac);
            if (MOM) {
                ma = fma(x[row], acc, ma);
                if (yjac) mb = fma(dinv[row] * acc, acc, mb);
            }
        }
    }
    if (MOM) spmv_moment_finish(ma, mb, mom_a, mom_b);
}

// ------------------------------------------------------------------------------------------------------
// Bulk-staged variant.  One warp owns a ring of D slots; slot = { double vals[CAP]; int cols[CAP] }.
// Tile t covers rows [t*RPT, (t+1)*RPT), RPT = 32/L; its nnz range [rp[row0], rp[row1]) is copied from the
// 16 B aligned element a0 = rp[row0] & ~3 on.  Tiles are dealt to warps round-robin so that at any time the
// grid works on one contiguous window of rows (keeps the gathered vector's working set in L2/L1).
//
// Per tile a lane holds a register fragment: its first U entries of the row (values, gathered x), the row's
// diagonal entry a_ii (1/a_ii is taken from the row itself: no dinv array is read) and the
// partial sum of any entries beyond U*L (long rows, summed when the fragment is loaded).  Once the fragment is in
// registers the slot is free and the copy of the warp's tile i+D is issued into it.  (Loading the fragment of tile
// i+1 before tile i is reduced was measured slower: it doubles the registers and halves the resident warps.)
// Three CTAs per SM is the optimum, not a register accident: forced to 64 registers (MINB = 4: 32 warps per SM, 92 bytes
// of spills) the same kernel takes 1790 us instead of 554 us on 320^3 and 103 us instead of 41 us on 128^3 -- four rings
// (196 KB of shared memory) leave the unified L1 about 30 KB, and the x gathers live on L1 hits (68 % at three CTAs).
template <int U>
struct SpmvFrag {
    double v[U], xv[U];
    double diag, rem, xrow, xprev;
};

template <int L, int D, int CAP, int WPC, bool MOM, int MINB = 3>
__global__ void __launch_bounds__(WPC * 32, MINB) spmv_bulk_kernel(int n, int nnz, const int* __restrict__ rp,
                                                             const int* __restrict__ ci, const double* __restrict__ va,
                                                             const double* __restrict__ x, double* __restrict__ y,
                                                             double* __restrict__ yjac, const double* __restrict__ xprev,
                                                             int mode, const ScgState* __restrict__ st, int num_tiles,
                                                             double* __restrict__ mom_a, double* __restrict__ mom_b) {
    // (the status test sits behind the ring prologue, after pdl_wait: the prologue touches only the constant CSR arrays)
    constexpr int RPT = 32 / L;
    constexpr int U = 8;  // entries per lane held in registers (rows up to 8 L entries need no remainder loop)
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* svals = reinterpret_cast<double*>(smem_raw) + (size_t)warp * D * CAP;
    int* scols = reinterpret_cast<int*>(smem_raw + (size_t)WPC * D * CAP * sizeof(double)) + (size_t)warp * D * CAP;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + (size_t)WPC * D * CAP * 12) + warp * D;

    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < D; d++) mbar_init(&bars[d], 1);
        mbar_fence_init();
    }
    __syncwarp();
    const uint64_t policy = l2_policy_evict_first();
    // 32-bit row / tile arithmetic (setup guarantees n + 64 < 2^31): keeps the kernel inside its 80-register budget
    const int GW = (int)gridDim.x * WPC;
    const int gw = (int)blockIdx.x * WPC + warp;
    if (!MOM && gw >= num_tiles) return;  // (the moment form ends in a block-wide reduction: every warp stays)
    const int my_tiles = (gw < num_tiles) ? (num_tiles - gw + GW - 1) / GW : 0;
    double ma = 0.0, mb = 0.0;  // moment partials (moment form only)
    const int g = lane % L;
    const bool jac = yjac != nullptr;

    // issue the copies of this warp's i-th tile into slot i % D; nz0/nz1 = its nnz range (valid in lane 0)
    auto issue = [&](int i, int nz0, int nz1) {
        const int sl = (int)(i % D);
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
                bulk_g2s(dv, va + a0, (uint32_t)cnt * 8u, &bars[sl], policy);
                bulk_g2s(dc, ci + a0, (uint32_t)cnt * 4u, &bars[sl], policy);
            } else {
                mbar_arrive(&bars[sl]);
            }
        }
        // ragged tail of the arrays (at most 3 elements of the whole matrix) by plain loads
        const int b_end = __shfl_sync(0xffffffffu, bulk_end, 0);
        const int b_a0 = __shfl_sync(0xffffffffu, a0, 0);
        const int b_nz1 = __shfl_sync(0xffffffffu, nz1, 0);
        if (b_end < b_nz1) {  // (warp-uniform; only the last tile of a matrix with nnz % 4 != 0 comes here)
            for (int e = b_end + lane; e < b_nz1; e += 32) {
                dv[e - b_a0] = va[e];
                dc[e - b_a0] = ci[e];
            }
            __syncwarp();  // other lanes read these entries in load_frag behind a per-lane mbarrier wait only
        }
    };
    auto tile_bounds = [&](int i, int& nz0, int& nz1) {  // lane 0 only
        const int t = gw + i * GW;
        const int row0 = t * RPT;
        int row1 = row0 + RPT;
        if (row1 > n) row1 = n;
        nz0 = rp[row0];
        nz1 = rp[row1];
    };
    auto row_of = [&](int i) { return (gw + i * GW) * RPT + lane / L; };

    // slot i % D -> registers (waits for the copy; reads this lane's entries; issues the x gather)
    auto load_frag = [&](int i, int lo, int hi, SpmvFrag<U>& f) {
        const int sl = (int)(i % D);
        const int row = row_of(i);
        const int a0 = __shfl_sync(0xffffffffu, lo, 0) & ~3;
        mbar_wait(&bars[sl], (uint32_t)((i / D) & 1));
        const double* sv = svals + sl * CAP - a0;
        const int* sc = scols + sl * CAP - a0;
        int c[U];
        f.diag = 0.0;
#pragma unroll
        for (int u = 0; u < U; u++) {
            const int kk = lo + g + u * L;
            const bool ok = kk < hi;
            c[u] = ok ? sc[kk] : -1;
            f.v[u] = ok ? sv[kk] : 0.0;
            if (c[u] == row) f.diag = f.v[u];
        }
#pragma unroll
        for (int u = 0; u < U; u++) f.xv[u] = (c[u] >= 0) ? x[c[u]] : 0.0;
        f.xrow = 0.0;
        f.xprev = 0.0;
        if ((MOM || (jac && mode != 0)) && row < n) {  // x_row: Chebyshev epilogue, and the moment x^T (A x)
            f.xrow = x[row];
            if (mode == 2) f.xprev = xprev[row];
        }
        double rem = 0.0;
        for (int k0 = lo + g + U * L; k0 < hi; k0 += U * L) {  // long rows only: further batches of U entries per lane
            int cc[U];
            double vv[U], xx[U];
#pragma unroll
            for (int u = 0; u < U; u++) {
                const int kk = k0 + u * L;
                const bool ok = kk < hi;
                cc[u] = ok ? sc[kk] : -1;
                vv[u] = ok ? sv[kk] : 0.0;
                if (cc[u] == row) f.diag = vv[u];
            }
#pragma unroll
            for (int u = 0; u < U; u++) xx[u] = (cc[u] >= 0) ? x[cc[u]] : 0.0;
#pragma unroll
            for (int u = 0; u < U; u++) rem = fma(vv[u], xx[u], rem);
        }
        f.rem = rem;
        __syncwarp();  // every lane has read the slot: it may be refilled
    };
    auto finish = [&](int i, const SpmvFrag<U>& f) {
        const int row = row_of(i);
        double acc = 0.0;
#pragma unroll
        for (int u = 0; u < U; u++) acc = fma(f.v[u], f.xv[u], acc);
        acc += f.rem;
        acc = group_sum<L>(acc);
        double d = f.diag;
        if (L > 1 && jac) d = group_sum<L>(d);  // exactly one lane of the group holds a_ii, the others 0
        if (g == 0 && row < n) {
            y[row] = acc;
            if (MOM) ma = fma(f.xrow, acc, ma);
            if (jac) {
                double z = __drcp_rn(d) * acc;  // = (1 / a_ii) * acc, the same two roundings as a dinv array
                if (MOM) mb = fma(z, acc, mb);
                if (mode == 1) z = z - f.xrow;
                else if (mode == 2) z = 2.0 * (z - f.xrow) - f.xprev;
                yjac[row] = z;
            }
        }
    };
    auto row_bounds = [&](int i, int& lo, int& hi) {
        lo = hi = 0;
        if (i < my_tiles) {
            const int row = row_of(i);
            if (row < n) { lo = rp[row]; hi = rp[row + 1]; }
        }
    };

    // prologue: fill the ring
    int nb0 = 0, nb1 = 0;  // nnz range of the next tile to issue (lane 0; fetched one step ahead)
    for (int i = 0; i < D && i < my_tiles; i++) {
        int a = 0, b = 0;
        if (lane == 0) tile_bounds(i, a, b);
        issue(i, a, b);
    }
    if (lane == 0 && D < my_tiles) tile_bounds(D, nb0, nb1);
    int lo_n, hi_n;  // per-row bounds of the next fragment to load (fetched one step ahead)
    row_bounds(0, lo_n, hi_n);

    // everything above read rowptr / colidx / vals only, which no kernel writes: under a programmatic dependent launch it
    // overlaps the tail of the previous kernel.  x, xprev, st and the outputs belong to the predecessor until here.
    pdl_wait();
    pdl_launch();
    if (st && st->status != SCG_RUNNING) {
        // not running: the copies already issued into this warp's ring must land before the block may exit
        for (int i = 0; i < D && i < my_tiles; i++) mbar_wait(&bars[i % D], 0u);
        return;
    }

    {
        SpmvFrag<U> cur;
        for (int i = 0; i < my_tiles; i++) {
            const int lo = lo_n, hi = hi_n;
            row_bounds(i + 1, lo_n, hi_n);
            load_frag(i, lo, hi, cur);
            if (i + D < my_tiles) {
                issue(i + D, nb0, nb1);
                if (lane == 0 && i + D + 1 < my_tiles) tile_bounds(i + D + 1, nb0, nb1);
            }
            finish(i, cur);
        }
    }
    if (MOM) spmv_moment_finish(ma, mb, mom_a, mom_b);
}

// max nnz over tiles of `rpt` rows (setup-time check for the bulk variant)
__global__ void tile_nnz_max_kernel(int64_t n, const int* __restrict__ rp, int rpt, int64_t num_tiles, int* __restrict__ out) {
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int m = 0;
    if (t < num_tiles) {
        int64_t r0 = t * rpt, r1 = r0 + rpt;
        if (r1 > n) r1 = n;
        m = rp[r1] - rp[r0];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(out, m);
}

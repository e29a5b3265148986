// common.cuh -- device helpers shared by the sm_100a kernels of the s-step PCG hot path.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define SCG_SMAX 16
#define SCG_WARP 32

// Device-resident solver state: everything the outer iteration needs that is not problem-sized.
// Written by the kernels, read by the host only through an async copy of the header.
struct ScgState {
    // ---- header (copied to the host when polling) ----
    int32_t status;      // -1 running, 0 converged, 2 breakdown
    int32_t k;           // outer iterations completed
    double rho;          // ||r||^2 after the last completed iteration
    double rho0;         // ||r_0||^2
    double rtol;         // stop when sqrt(rho) < rtol * sqrt(rho0)  (Alg. 3 l.31)
    // ---- small dense state ----
    double W[SCG_SMAX * SCG_SMAX];      // W of the previous outer iteration (P^T A P), row-major
    double beta[SCG_SMAX * SCG_SMAX];
    double alpha[SCG_SMAX];
    double M[SCG_SMAX * SCG_SMAX];
    double C[SCG_SMAX * SCG_SMAX];
    double m[SCG_SMAX];
    double Lw[SCG_SMAX * SCG_SMAX];     // Cholesky factor of W (lower triangle, row-major): the next iteration's beta solve reuses it
    // ---- moment form (option "form" = 1): mu^0 = R_1^T r from the update / init kernel, the 2s moments of the last MPK
    double mu0;
    double vm[2 * SCG_SMAX];
    // ---- cross-block finish tickets (reset by the last block, so graphs can be replayed) ----
    unsigned int ticket_gram;
    unsigned int ticket_update;
    unsigned int ticket_init;
    // grid barrier of the resident (cooperative) kernel, zeroed before each launch: arrival counter and, in another
    // 128-byte line (the pollers must not queue behind the arriving atomics), the generation flag the last arriver sets
    unsigned int grid_bar;
    unsigned int grid_pad[31];
    unsigned int grid_flag;
};
#define SCG_RUNNING (-1)

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Fixed-order sum of p[0 .. cnt) by one warp (cross-block finishes): lane-strided with eight independent accumulators,
// the eight loads of a pass issued together so that their L2 round trips overlap (a few hundred partials cost two
// round trips instead of five); the order depends only on cnt, so the result is reproducible run to run.
__device__ __forceinline__ double warp_sum_array(const double* p, int cnt, int lane) {
    double a[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    int b = lane;
    for (; b + 224 < cnt; b += 256) {
        double v[8];
#pragma unroll
        for (int k = 0; k < 8; k++) v[k] = __ldcg(p + b + 32 * k);
#pragma unroll
        for (int k = 0; k < 8; k++) a[k] += v[k];
    }
    {
        double v[8];
#pragma unroll
        for (int k = 0; k < 8; k++) v[k] = (b + 32 * k < cnt) ? __ldcg(p + b + 32 * k) : 0.0;
#pragma unroll
        for (int k = 0; k < 8; k++) a[k] += v[k];
    }
    double v = ((a[0] + a[1]) + (a[2] + a[3])) + ((a[4] + a[5]) + (a[6] + a[7]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// The same sums for K arrays p, p + stride, ... at once (entries beyond kvalid give 0): per array the order of
// warp_sum_array, bit for bit, but the loads of all K arrays of a pass are in flight together, so a warp that owns several
// entries of a cross-block finish pays the L2 round trips once instead of K times.
template <int K>
__device__ __forceinline__ void warp_sum_arrays(const double* p, int64_t stride, int kvalid, int cnt, int lane, double (&out)[K]) {
    double a[K][8];
#pragma unroll
    for (int q = 0; q < K; q++)
#pragma unroll
        for (int k = 0; k < 8; k++) a[q][k] = 0.0;
    int b = lane;
    for (; b + 224 < cnt; b += 256) {
        double v[K][8];
#pragma unroll
        for (int q = 0; q < K; q++)
#pragma unroll
            for (int k = 0; k < 8; k++) v[q][k] = (q < kvalid) ? __ldcg(p + q * stride + b + 32 * k) : 0.0;
#pragma unroll
        for (int q = 0; q < K; q++)
#pragma unroll
            for (int k = 0; k < 8; k++) a[q][k] += v[q][k];
    }
    {
        double v[K][8];
#pragma unroll
        for (int q = 0; q < K; q++)
#pragma unroll
            for (int k = 0; k < 8; k++) v[q][k] = (q < kvalid && b + 32 * k < cnt) ? __ldcg(p + q * stride + b + 32 * k) : 0.0;
#pragma unroll
        for (int q = 0; q < K; q++)
#pragma unroll
            for (int k = 0; k < 8; k++) a[q][k] += v[q][k];
    }
#pragma unroll
    for (int q = 0; q < K; q++) {
        double v = ((a[q][0] + a[q][1]) + (a[q][2] + a[q][3])) + ((a[q][4] + a[q][5]) + (a[q][6] + a[q][7]));
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        out[q] = v;
    }
}

// Sums over the 32 lanes of K values per lane at once, by recursive halving: in the step with lane offset OFF a lane keeps
// one half of its values and hands the other half to its partner, so the values per lane halve while the lanes per sum
// double -- ceil(K/2) + ceil(K/4) + ... shuffles (37 for K = 36) instead of 5 K (180) for K separate butterfly sums.  On
// return v[t], t < nvalid (<= warp_reduce_many_count(K)), holds the complete sum of entry `base + t`; every entry is held by
// exactly one lane of the warp (halves that are empty padding are tracked by nvalid); the summation order depends only on K.
__host__ __device__ constexpr int warp_reduce_many_count(int k) {
    for (int step = 0; step < 5; step++) k = (k + 1) / 2;
    return k;
}
template <int KC, int OFF, int K>
__device__ __forceinline__ void warp_reduce_many_step(double (&v)[K], int lane, int& base, int& nvalid) {
    if constexpr (OFF >= 1) {
        constexpr int H = (KC + 1) / 2;
        const bool up = (lane & OFF) != 0;
#pragma unroll
        for (int i = 0; i < H; i++) {
            const double lo = v[i];
            const double hi = (i + H < KC) ? v[i + H] : 0.0;
            const double send = up ? lo : hi;
            const double keep = up ? hi : lo;
            v[i] = keep + __shfl_xor_sync(0xffffffffu, send, OFF);
        }
        if (up) { base += H; nvalid = nvalid > H ? nvalid - H : 0; }  // the upper half: slots [H, KC) of the old numbering
        else nvalid = nvalid < H ? nvalid : H;
        warp_reduce_many_step<H, OFF / 2, K>(v, lane, base, nvalid);
    }
}
template <int K>
__device__ __forceinline__ int warp_reduce_many(double (&v)[K], int lane, int& nvalid) {
    int base = 0;
    nvalid = K;
    warp_reduce_many_step<K, 16, K>(v, lane, base, nvalid);
    return base;
}

template <int L>
__device__ __forceinline__ double group_sum(double v) {
#pragma unroll
    for (int o = L / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---- mbarrier + 1-D bulk async copy (TMA engine, cp.async.bulk) -------------------------------------
// ---- programmatic dependent launch (sm_90+): the kernels of one outer iteration are chained with the launch attribute
// cudaLaunchAttributeProgrammaticStreamSerialization, so the blocks of kernel k+1 may become resident (and run whatever
// does not depend on kernel k) while kernel k drains.  pdl_wait() returns once every prerequisite grid has completed and
// its writes are visible -- nothing written by (or still read by) the predecessor may be touched before it; it is a
// no-op for a launch without the attribute.  pdl_launch() lets the next kernel's blocks be scheduled.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// one non-blocking probe of the phase with the given parity
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// global -> shared bulk copy; dst/src 16 B aligned, bytes a multiple of 16; completes on `bar` (complete_tx).
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar,
                                         uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
// the same without a cache hint (data that is re-read soon: default L2 policy)
__device__ __forceinline__ void bulk_g2s_nohint(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// shared -> global bulk copy (TMA store), tracked by the issuing thread's bulk async-group
__device__ __forceinline__ void bulk_s2g(void* dst_gmem, const void* src_smem, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// all bulk stores of this thread have finished READING shared memory (the source may be reused)
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
// ... and have been written to global memory
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// streaming (read-once) 128-bit and 64-bit global loads
__device__ __forceinline__ double2 ldg_stream2(const double* p) {
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
// read-only load that allocates in L1 (re-read by the other warps of the CTA); asm volatile keeps a batch of loads
// together in program order, ahead of the arithmetic that consumes them
__device__ __forceinline__ double ldg_nc(const double* p) {
    double v;
    asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ double ldg_stream(const double* p) {
    double v;
    asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}

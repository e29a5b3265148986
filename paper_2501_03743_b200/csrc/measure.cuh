// measure.cuh -- measurement aids of bench.py's `roofline` object (not on the hot path): hand-written streaming kernels
// that give the READ-side and the copy bandwidth of this box with the same load instructions the hot kernels use, so
// that the SpMV (87 % reads) and the Gram kernel (99.9 % reads) can be set against a read-only wall instead of the
// read+write copy peak of MEASURED_PEAKS.json.  A buffer of `bytes` bytes is swept `passes` times inside one launch
// (passes > 1 on a buffer smaller than L2 measures the L2-hit bandwidth, which bounds what an L2-served matrix-powers
// pass could gain).
//   variant 0: 128-bit ld.global.nc.L1::no_allocate (the Gram / update kernels' loads)
//   variant 1, 3, 4, 5: cp.async.bulk global -> shared through per-warp mbarrier rings of different shapes -- the number of
//              bulk copies an SM keeps in flight decides: 48 x 4 KB, 96 x 2 KB, 24 x 8 KB, 32 x 4 KB
//   variant 2: 128-bit copy (read + write), bytes counted twice
#pragma once
#include "common.cuh"

__global__ void __launch_bounds__(256, 4)
measure_read_ldg_kernel(const double2* __restrict__ src, int64_t n16, int passes, double* __restrict__ sink) {
    double acc = 0.0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x * 4;
    for (int p = 0; p < passes; p++) {
        for (int64_t i = ((int64_t)blockIdx.x * blockDim.x) * 4 + threadIdx.x; i < n16; i += stride) {
            double2 v[4];
#pragma unroll
            for (int u = 0; u < 4; u++) {
                const int64_t k = i + (int64_t)u * blockDim.x;
                v[u] = (k < n16) ? ldg_stream2(reinterpret_cast<const double*>(src + k)) : make_double2(0.0, 0.0);
            }
#pragma unroll
            for (int u = 0; u < 4; u++) acc += v[u].x + v[u].y;
        }
    }
    if (acc == 1.2345e301) sink[0] = acc;  // keeps the loads alive; never true for the zero-filled buffer
}

// WPC warps per CTA; each warp owns a ring of D slots of CHUNK bytes and walks its share of the buffer
template <int D, int CHUNK, int WPC>
__global__ void __launch_bounds__(WPC * 32, 3)
measure_read_bulk_kernel(const unsigned char* __restrict__ src, int64_t nchunks, int passes, double* __restrict__ sink) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char* ring = smem_raw + (size_t)warp * D * CHUNK;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + (size_t)WPC * D * CHUNK) + warp * D;
    if (lane == 0) {
        for (int d = 0; d < D; d++) mbar_init(&bars[d], 1);
        mbar_fence_init();
    }
    __syncwarp();
    const uint64_t policy = l2_policy_evict_first();
    const int64_t GW = (int64_t)gridDim.x * WPC, gw = (int64_t)blockIdx.x * WPC + warp;
    const int64_t per_pass = (gw < nchunks) ? (nchunks - gw + GW - 1) / GW : 0;
    const int64_t mine = per_pass * passes;
    double acc = 0.0;
    auto chunk_of = [&](int64_t i) { return gw + (i % per_pass) * GW; };
    for (int64_t i = 0; i < D && i < mine; i++) {
        if (lane == 0) {
            mbar_expect_tx(&bars[i % D], CHUNK);
            if (passes > 1) bulk_g2s_nohint(ring + (i % D) * CHUNK, src + chunk_of(i) * CHUNK, CHUNK, &bars[i % D]);
            else bulk_g2s(ring + (i % D) * CHUNK, src + chunk_of(i) * CHUNK, CHUNK, &bars[i % D], policy);
        }
    }
    for (int64_t i = 0; i < mine; i++) {
        const int sl = (int)(i % D);
        mbar_wait(&bars[sl], (uint32_t)((i / D) & 1));
        acc += reinterpret_cast<const double*>(ring + sl * CHUNK)[lane];  // one touch per slot: the data did arrive
        __syncwarp();
        if (i + D < mine && lane == 0) {
            fence_proxy_async_smem();
            mbar_expect_tx(&bars[sl], CHUNK);
            if (passes > 1) bulk_g2s_nohint(ring + sl * CHUNK, src + chunk_of(i + D) * CHUNK, CHUNK, &bars[sl]);
            else bulk_g2s(ring + sl * CHUNK, src + chunk_of(i + D) * CHUNK, CHUNK, &bars[sl], policy);
        }
    }
    if (acc == 1.2345e301) sink[0] = acc;
}

__global__ void __launch_bounds__(256, 4)
measure_copy_kernel(const double2* __restrict__ src, double2* __restrict__ dst, int64_t n16, int passes) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x * 4;
    for (int p = 0; p < passes; p++) {
        for (int64_t i = ((int64_t)blockIdx.x * blockDim.x) * 4 + threadIdx.x; i < n16; i += stride) {
            double2 v[4];
#pragma unroll
            for (int u = 0; u < 4; u++) {
                const int64_t k = i + (int64_t)u * blockDim.x;
                v[u] = (k < n16) ? ldg_stream2(reinterpret_cast<const double*>(src + k)) : make_double2(0.0, 0.0);
            }
#pragma unroll
            for (int u = 0; u < 4; u++) {
                const int64_t k = i + (int64_t)u * blockDim.x;
                if (k < n16) dst[k] = v[u];
            }
        }
    }
}

// launch of one bulk-read shape on at most ctas_per_sm CTAs per SM
template <int D, int CHUNK, int WPC>
cudaError_t launch_measure_bulk(int num_sms, int ctas_per_sm, cudaStream_t sm, const unsigned char* src, int64_t bytes, int passes, double* sink) {
    const size_t smem = (size_t)WPC * D * CHUNK + (size_t)WPC * D * 8;
    auto k = measure_read_bulk_kernel<D, CHUNK, WPC>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int occ = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, WPC * 32, smem);
    if (e != cudaSuccess) return e;
    if (occ > ctas_per_sm) occ = ctas_per_sm;
    if (occ < 1) return cudaErrorInvalidConfiguration;
    k<<<occ * num_sms, WPC * 32, smem, sm>>>(src, bytes / CHUNK, passes, sink);
    return cudaGetLastError();
}

// tile_pipe.cuh -- producer/consumer tile pipeline for the block kernels (Gram, update) at larger s.
//
// Why: with s >= 5 a thread's registers are taken by accumulators / row data, so too few bytes are in flight
// per SM to cover the HBM latency (profiles/r01a: gram<8> 64 %, update<8> 80 % of the copy peak).  Here the bytes
// in flight live in shared memory instead: a producer warp streams row tiles of every operand with the TMA engine
// (cp.async.bulk 1-D, mbarrier complete_tx) into a D-slot ring, the consumer warps compute from shared memory.
//
// One warp sustains only ~15 GB/s of bulk copies (measured), so NPW producer warps share the tiles round-robin
// (tile i is filled by producer i % NPW).  The mbarrier waits are parity waits, which cannot tell phase k from phase
// k-2: a producer must never get two phases ahead of a slot, which holds iff NPW <= D.
//
// A tile is T consecutive rows.  Each operand contributes contiguous global SEGMENTS (a column slice of a
// column-major block, the T*s doubles of an interleaved block, a slice of a vector).  Bulk copies need 16-byte
// aligned addresses and sizes, segments are only 8-byte aligned, so a segment is copied from its address rounded
// DOWN to 16 bytes up to its end rounded UP (at most one neighbouring double on each side, always inside the same
// allocation); the consumer skips `shift` (0 or 1) leading doubles.  If the rounded-up end would cross the end of
// the allocation the last double is fetched by a plain load instead.
#pragma once
#include "common.cuh"

struct TileSeg {
    const double* g;        // first wanted double in global memory
    const double* buf_end;  // one past the allocation the segment lives in
    double* dst;            // 16-byte aligned shared-memory sub-buffer, capacity cnt + 2 doubles
    int cnt;                // wanted doubles
};

// element k of the segment lands at dst[seg_shift(g) + k]
__device__ __forceinline__ int seg_shift(const double* g) { return (int)(((uintptr_t)g >> 3) & 1); }

// bytes the bulk copy of this segment moves (0 = nothing to copy); `tail` = last double needs a plain load
__device__ __forceinline__ uint32_t seg_plan(const TileSeg& sg, bool& tail) {
    tail = false;
    if (sg.cnt <= 0) return 0;
    const uintptr_t a = (uintptr_t)sg.g, a0 = a & ~(uintptr_t)15;
    uintptr_t e1 = (a + 8u * (uintptr_t)sg.cnt + 15) & ~(uintptr_t)15;
    if (e1 > (uintptr_t)sg.buf_end) { e1 -= 16; tail = true; }
    return e1 > a0 ? (uint32_t)(e1 - a0) : 0u;
}

// Producer warp, all 32 lanes: fill one slot with `nseg` segments described by make_seg(c) and arm `full`.
// The slot must already be free (its `empty` phase waited for by the caller).
template <class MakeSeg>
__device__ __forceinline__ void tile_fill(int nseg, MakeSeg make_seg, uint64_t* full, uint64_t policy, int lane) {
    uint32_t bytes = 0;
    for (int c = lane; c < nseg; c += 32) {
        const TileSeg sg = make_seg(c);
        bool tail;
        bytes += seg_plan(sg, tail);
        if (tail) sg.dst[seg_shift(sg.g) + sg.cnt - 1] = sg.g[sg.cnt - 1];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) bytes += __shfl_xor_sync(0xffffffffu, bytes, o);
    __syncwarp();  // the tail stores of the other lanes are ordered before lane 0's releasing arrive below
    if (lane == 0) {
        fence_proxy_async_smem();  // consumers' generic reads of this slot are ordered before the async writes
        mbar_expect_tx(full, bytes);  // one arrival + the transaction bytes (release: publishes the tail stores)
    }
    __syncwarp();
    for (int c = lane; c < nseg; c += 32) {
        const TileSeg sg = make_seg(c);
        bool tail;
        const uint32_t b = seg_plan(sg, tail);
        if (b) bulk_g2s(sg.dst, (const void*)((uintptr_t)sg.g & ~(uintptr_t)15), b, full, policy);
    }
}

// reorder.cuh -- setup-time symmetric reordering for gather locality (option "reorder").
//
// Why: the SpMV of the matrix-powers kernel (Alg. 4) gathers R_j(col) for every non-zero.  When the
// rows of A are numbered without locality (BASELINE.json config 5: "rows randomly permuted to break locality") and the
// vector is larger than L2, every 8-byte gather costs a 64-byte DRAM access: ncu shows 7.0 GB of DRAM reads per launch
// against 1.9 GB of algorithmic traffic (profiles/r01c_tuned_path.md).  The paper's own matrices come from a
// structured grid and its distributed SpMV relies on a contiguous row-block decomposition with few halo entries
// (PAPER.md:206); a symmetric permutation A' = Pi A Pi^T, b' = Pi b leaves every CG / s-step iterate unchanged in exact
// arithmetic (the Jacobi preconditioner commutes with it) and only changes the order of the Gram sums.
//
// What: Cuthill-McKee numbering on the device.  A pseudo-peripheral root is found with one level-synchronous BFS
// (farthest level, smallest index); the numbering BFS then appends level after level, each level sorted by
// (rank of the first-numbered parent, original index) -- one 64-bit radix sort per level (cub::DeviceRadixSort, a
// library sort used as a setup step), so the result is deterministic whatever order the atomics discover nodes in.
// Neighbours of consecutively numbered rows end up consecutively numbered in the adjacent level: the gathers of a
// warp fall into a few sectors again and the working set (about three levels) stays in L2.
// Then the CSR arrays are permuted into an owned copy; b and x0 are permuted on the way in, x on the way out.
#pragma once
#include <cub/cub.cuh>

#include <climits>

#include "common.cuh"

namespace scg_reorder {

__global__ void fill_int_kernel(int* __restrict__ p, int v, int64_t n) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) p[i] = v;
}

// share of the off-diagonal entries whose column is further than `window` rows away from the row
__global__ void far_entries_kernel(int64_t n, const int* __restrict__ rp, const int* __restrict__ ci, int window,
                                   unsigned long long* __restrict__ far) {
    const int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned int cnt = 0;
    if (row < n)
        for (int k = rp[row]; k < rp[row + 1]; k++) {
            const int64_t d = (int64_t)ci[k] - row;
            if (d > window || -d > window) cnt++;
        }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(far, (unsigned long long)cnt);
}

// One BFS level.  frontier[0..nf) = the nodes of level L, frontier[t] has rank base + t.  Unseen neighbours get level
// L + 1 and are appended to `next` (order = whatever the atomics give; fixed later by the sort).  minpar (may be null:
// root search) receives the smallest rank among the level-L parents of every level-(L+1) node.
__global__ void bfs_expand_kernel(int nf, const int* __restrict__ frontier, int base, int L, const int* __restrict__ rp,
                                  const int* __restrict__ ci, int* __restrict__ level, int* __restrict__ minpar,
                                  int* __restrict__ next, int* __restrict__ next_cnt) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nf) return;
    const int u = frontier[t], ru = base + t;
    for (int k = rp[u]; k < rp[u + 1]; k++) {
        const int v = ci[k];
        if (v == u) continue;
        int old = level[v];
        if (old == -1) old = atomicCAS(&level[v], -1, L + 1);
        if (old == -1) next[atomicAdd(next_cnt, 1)] = v;
        if (minpar && (old == -1 || old == L + 1)) atomicMin(&minpar[v], ru);
    }
}

__global__ void make_keys_kernel(int nf, const int* __restrict__ nodes, const int* __restrict__ minpar, int base_prev, int vbits,
                                 unsigned long long* __restrict__ keys) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nf) return;
    const int v = nodes[t];
    keys[t] = ((unsigned long long)(unsigned int)(minpar[v] - base_prev) << vbits) | (unsigned int)v;
}

__global__ void place_sorted_kernel(int nf, const unsigned long long* __restrict__ keys, int vbits, int base,
                                    int* __restrict__ perm, int* __restrict__ rank) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nf) return;
    const int v = (int)(keys[t] & ((1ull << vbits) - 1ull));
    perm[base + t] = v;
    rank[v] = base + t;
}

__global__ void min_of_list_kernel(int nf, const int* __restrict__ list, int* __restrict__ out) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < nf) atomicMin(out, list[t]);
}

__global__ void first_unseen_kernel(int n, const int* __restrict__ level, int* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && level[i] == -1) atomicMin(out, i);
}

// nodes not numbered yet (level == -1) keep their relative order and go to the end: flag -> exclusive scan -> place
__global__ void flag_unseen_kernel(int n, const int* __restrict__ level, int* __restrict__ flag) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) flag[i] = (level[i] == -1) ? 1 : 0;
}
__global__ void place_unseen_kernel(int n, const int* __restrict__ level, const int* __restrict__ offs, int base,
                                    int* __restrict__ perm, int* __restrict__ rank) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && level[i] == -1) { perm[base + offs[i]] = i; rank[i] = base + offs[i]; }
}

__global__ void set_root_kernel(int root, int pos, int* __restrict__ level, int* __restrict__ perm, int* __restrict__ rank) {
    level[root] = 0;
    if (perm) { perm[pos] = root; rank[root] = pos; }
}

__global__ void row_len_kernel(int n, const int* __restrict__ perm, const int* __restrict__ rp, int* __restrict__ len) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { const int o = perm[i]; len[i] = rp[o + 1] - rp[o]; }
    if (i == n) len[n] = 0;
}

// new row i = old row perm[i]; columns renumbered by rank; 8 lanes per row
__global__ void permute_csr_kernel(int n, const int* __restrict__ perm, const int* __restrict__ rank, const int* __restrict__ rp,
                                   const int* __restrict__ ci, const double* __restrict__ va, const int* __restrict__ rp2,
                                   int* __restrict__ ci2, double* __restrict__ va2) {
    const int64_t gt = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t i = gt >> 3;
    const int g = (int)(gt & 7);
    if (i >= n) return;
    const int o = perm[i];
    const int src = rp[o], len = rp[o + 1] - src, dst = rp2[i];
    for (int k = g; k < len; k += 8) {
        ci2[dst + k] = rank[ci[src + k]];
        va2[dst + k] = va[src + k];
    }
}

__global__ void gather_vec_kernel(int64_t n, const int* __restrict__ perm, const double* __restrict__ src, double* __restrict__ dst) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[perm[i]];
}
__global__ void scatter_vec_kernel(int64_t n, const int* __restrict__ perm, const double* __restrict__ src, double* __restrict__ dst) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[perm[i]] = src[i];
}

inline unsigned blocks_for(int64_t n, int bs = 256) { return (unsigned)((n + bs - 1) / bs); }
inline int bits_for(unsigned int maxval) {
    int b = 1;
    while (b < 32 && (maxval >> b)) b++;
    return b;
}

#define SCG_RCK(call)                        \
    do {                                     \
        cudaError_t e_ = (call);             \
        if (e_ != cudaSuccess) return e_;    \
    } while (0)

// Cuthill-McKee numbering of the graph of (rp, ci).  perm[new] = old, rank[old] = new (device, n ints each).
// After `max_components` components (a matrix with very many tiny components would otherwise cost one BFS each) the
// nodes still unnumbered are appended in their original order.  *done = false only on a CUDA error.
// levels_out / comps_out: statistics (comps_out counts the components numbered by BFS).
inline cudaError_t cuthill_mckee(int n, const int* rp, const int* ci, cudaStream_t sm, int* perm, int* rank, bool* done,
                                 int* levels_out, int* comps_out, int max_components = 64) {
    *done = false;
    int *level = nullptr, *scratch = nullptr, *minpar = nullptr, *cnt = nullptr;
    unsigned long long *keys = nullptr, *keys2 = nullptr;
    void* tmp = nullptr;
    size_t tmp_bytes = 0;
    auto cleanup = [&]() {
        cudaFree(level); cudaFree(scratch); cudaFree(minpar); cudaFree(cnt); cudaFree(keys); cudaFree(keys2); cudaFree(tmp);
    };
    auto body = [&]() -> cudaError_t {
        SCG_RCK(cudaMalloc(&level, sizeof(int) * (size_t)n));
        SCG_RCK(cudaMalloc(&scratch, sizeof(int) * (size_t)n));
        SCG_RCK(cudaMalloc(&minpar, sizeof(int) * (size_t)n));
        SCG_RCK(cudaMalloc(&cnt, sizeof(int) * 4));
        SCG_RCK(cudaMalloc(&keys, sizeof(unsigned long long) * (size_t)n));
        SCG_RCK(cudaMalloc(&keys2, sizeof(unsigned long long) * (size_t)n));
        SCG_RCK(cub::DeviceRadixSort::SortKeys(nullptr, tmp_bytes, keys, keys2, n, 0, 64, sm));
        SCG_RCK(cudaMalloc(&tmp, tmp_bytes));
        const unsigned fb = 1184;
        fill_int_kernel<<<fb, 256, 0, sm>>>(level, -1, n);
        fill_int_kernel<<<fb, 256, 0, sm>>>(scratch, -1, n);
        fill_int_kernel<<<fb, 256, 0, sm>>>(minpar, INT_MAX, n);
        int* fa = reinterpret_cast<int*>(keys);   // frontier ping-pong of the root search (the key buffers are free then)
        int* fbuf = reinterpret_cast<int*>(keys2);
        const int vbits = bits_for((unsigned)(n - 1));
        int placed = 0, comps = 0, levels = 0, h = 0;
        while (placed < n) {
            if (comps >= max_components) {  // append the rest in index order
                int* flag = reinterpret_cast<int*>(keys);
                int* offs = reinterpret_cast<int*>(keys2);
                flag_unseen_kernel<<<blocks_for(n), 256, 0, sm>>>(n, level, flag);
                size_t tb = tmp_bytes;
                size_t need = 0;
                SCG_RCK(cub::DeviceScan::ExclusiveSum(nullptr, need, flag, offs, n, sm));
                if (need > tb) {
                    cudaFree(tmp);
                    tmp = nullptr;
                    SCG_RCK(cudaMalloc(&tmp, need));
                    tmp_bytes = tb = need;
                }
                SCG_RCK(cub::DeviceScan::ExclusiveSum(tmp, tb, flag, offs, n, sm));
                place_unseen_kernel<<<blocks_for(n), 256, 0, sm>>>(n, level, offs, placed, perm, rank);
                placed = n;
                break;
            }
            // ---- a start node of this component: the smallest unnumbered index
            int start = 0;
            if (comps > 0) {
                fill_int_kernel<<<1, 32, 0, sm>>>(cnt + 1, INT_MAX, 1);
                first_unseen_kernel<<<blocks_for(n), 256, 0, sm>>>(n, level, cnt + 1);
                SCG_RCK(cudaMemcpyAsync(&start, cnt + 1, sizeof(int), cudaMemcpyDeviceToHost, sm));
                SCG_RCK(cudaStreamSynchronize(sm));
            }
            // ---- pseudo-peripheral root: BFS on the scratch levels, smallest index of the last level
            set_root_kernel<<<1, 1, 0, sm>>>(start, 0, scratch, nullptr, nullptr);
            SCG_RCK(cudaMemcpyAsync(fa, &start, sizeof(int), cudaMemcpyHostToDevice, sm));
            int nf = 1;
            int *cur = fa, *nxt = fbuf;
            for (int L = 0;; L++) {
                SCG_RCK(cudaMemsetAsync(cnt, 0, sizeof(int), sm));
                bfs_expand_kernel<<<blocks_for(nf), 256, 0, sm>>>(nf, cur, 0, L, rp, ci, scratch, nullptr, nxt, cnt);
                SCG_RCK(cudaMemcpyAsync(&h, cnt, sizeof(int), cudaMemcpyDeviceToHost, sm));
                SCG_RCK(cudaStreamSynchronize(sm));
                if (h == 0) break;
                nf = h;
                int* t = cur; cur = nxt; nxt = t;
            }
            int root = start;
            fill_int_kernel<<<1, 32, 0, sm>>>(cnt + 1, INT_MAX, 1);
            min_of_list_kernel<<<blocks_for(nf), 256, 0, sm>>>(nf, cur, cnt + 1);
            SCG_RCK(cudaMemcpyAsync(&root, cnt + 1, sizeof(int), cudaMemcpyDeviceToHost, sm));
            SCG_RCK(cudaStreamSynchronize(sm));
            // ---- numbering BFS from the root: the frontier of level L is perm[base .. base + nf)
            set_root_kernel<<<1, 1, 0, sm>>>(root, placed, level, perm, rank);
            int base = placed;
            nf = 1;
            placed += 1;
            for (int L = 0;; L++) {
                levels++;
                SCG_RCK(cudaMemsetAsync(cnt, 0, sizeof(int), sm));
                int* next = reinterpret_cast<int*>(keys2);  // discovery list; consumed by make_keys before the sort overwrites it
                bfs_expand_kernel<<<blocks_for(nf), 256, 0, sm>>>(nf, perm + base, base, L, rp, ci, level, minpar, next, cnt);
                SCG_RCK(cudaMemcpyAsync(&h, cnt, sizeof(int), cudaMemcpyDeviceToHost, sm));
                SCG_RCK(cudaStreamSynchronize(sm));
                if (h == 0) break;
                make_keys_kernel<<<blocks_for(h), 256, 0, sm>>>(h, next, minpar, base, vbits, keys);
                const int end_bit = vbits + bits_for((unsigned)(nf - 1));
                size_t tb = tmp_bytes;
                SCG_RCK(cub::DeviceRadixSort::SortKeys(tmp, tb, keys, keys2, h, 0, end_bit, sm));
                place_sorted_kernel<<<blocks_for(h), 256, 0, sm>>>(h, keys2, vbits, placed, perm, rank);
                base = placed;
                nf = h;
                placed += h;
            }
            comps++;
        }
        SCG_RCK(cudaGetLastError());
        SCG_RCK(cudaStreamSynchronize(sm));
        *done = true;
        if (levels_out) *levels_out = levels;
        if (comps_out) *comps_out = comps;
        return cudaSuccess;
    };
    const cudaError_t e = body();
    cudaStreamSynchronize(sm);
    cleanup();
    return e;
}

// A' = Pi A Pi^T into caller-allocated arrays (rp2: n + 1, ci2 / va2: nnz).
inline cudaError_t permute_csr(int n, int nnz, const int* perm, const int* rank, const int* rp, const int* ci, const double* va,
                               int* rp2, int* ci2, double* va2, cudaStream_t sm) {
    int* len = nullptr;
    void* tmp = nullptr;
    size_t tb = 0;
    SCG_RCK(cudaMalloc(&len, sizeof(int) * ((size_t)n + 1)));
    row_len_kernel<<<blocks_for((int64_t)n + 1), 256, 0, sm>>>(n, perm, rp, len);
    cudaError_t e = cub::DeviceScan::ExclusiveSum(nullptr, tb, len, rp2, n + 1, sm);
    if (e == cudaSuccess) e = cudaMalloc(&tmp, tb);
    if (e == cudaSuccess) e = cub::DeviceScan::ExclusiveSum(tmp, tb, len, rp2, n + 1, sm);
    if (e == cudaSuccess) {
        permute_csr_kernel<<<blocks_for((int64_t)n * 8), 256, 0, sm>>>(n, perm, rank, rp, ci, va, rp2, ci2, va2);
        e = cudaGetLastError();
    }
    cudaStreamSynchronize(sm);
    cudaFree(len);
    cudaFree(tmp);
    (void)nnz;
    return e;
}

}  // namespace scg_reorder

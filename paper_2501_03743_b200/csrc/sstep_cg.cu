// sstep_cg.cu -- C ABI (include/sstep_cg.h) of the B200-native s-step PCG hot path: handle, setup,
// CUDA-graph capture of one outer iteration, the solve loop, and the test hooks.  sm_100a only, no CPU fallback.
#include "sstep_cg.h"

#include <chrono>
#include <cstdio>
#include <cstring>
#include <string>

#include "common.cuh"
#include "gram.cuh"
#include "gram_tma.cuh"
#include "measure.cuh"
#include "moment.cuh"
#include "pcg.cuh"
#include "reorder.cuh"
#include "resident.cuh"
#include "spmv.cuh"
#include "spmv_cta.cuh"
#include "update.cuh"
#include "update_tma.cuh"

namespace {

struct Header {  // mirrors the first fields of ScgState
    int32_t status, k;
    double rho, rho0, rtol;
};

// bulk-staged SpMV shapes: nnz capacity of one warp tile / warps per CTA.  256 x 8 is the thread-per-row shape of the
// 7-point configs; the two larger tiles keep FEW lanes per row for longer rows (27-point: L = 2 -> 16 rows x 27, L = 1 ->
// 32 rows x 27 per tile), because consecutive rows under the same lane index gather consecutive x entries.
constexpr int BULK_CAP = 256, BULK_WPC = 8;
// L = 2, depth 2 (27-point 160^3).  Bytes in flight decide: 8 warps x 2 CTAs on 512-entry slots 257 us per launch,
// 10 warps x 2 CTAs on 448-entry slots (40 slots = 208 KB of copies in flight per SM, the most that fits) 230 us = 97 %
// of the copy peak.  Measured on the way: 6 warps x 2 CTAs 313 us; 4 warps x 4 CTAs 254 us per launch but a slower outer
// iteration; 8 warps on 448-entry slots (60 instead of 28 KB of L1) 256 us -- L1 is not the limit here.
constexpr int BULK_CAP2 = 448, BULK_WPC2 = 10;    // tiles up to 445 entries (16 rows x 27)
constexpr int BULK_CAP2B = 512, BULK_WPC2B = 8;   // tiles up to 509 entries (16 rows x 31)
constexpr int BULK_CAP1 = 1024, BULK_WPC1 = 4;    // L = 1, depth 2
constexpr size_t bulk_smem_for(int D, int cap, int wpc) { return (size_t)wpc * D * cap * 12 + (size_t)wpc * D * 8; }
// CTA-pipelined SpMV (spmv_cta.cuh), thread-per-row matrices: tiles of 256 rows, stage capacity 1800 entries (a 7-point
// tile holds <= 1792; three stages x three CTAs = 194 KB of shared memory per SM, ~33 KB left for L1)
constexpr int CTA_TR = 256, CTA_CAPT = 1800;
// two lanes per row (mean rows of 16-32 entries: the 27-point config): tiles of 128 rows (8 consumer warps x 16 rows), stage
// capacity 3472 entries (27 x 128 = 3456), 14 entries per lane in registers, two stages x two CTAs = 167 KB per SM
constexpr int CTA2_TR = 128, CTA2_CAPT = 3472, CTA2_U = 14;
// ... and, when no moment partials ride on the SpMV (Gram form), tiles of 96 rows on THREE CTAs per SM: 208.5 instead of 213 us
// per launch on 27-point 160^3 (the instantiation with the moment epilogue spills at that register budget: 314 us)
constexpr int CTA2B_TR = 96, CTA2B_CAPT = 2608;

}  // namespace

struct sstep_cg {
    int device = 0;
    cudaStream_t stream = nullptr;      // borrowed
    cudaStream_t cap_stream = nullptr;  // owned, used only to capture the graph
    int num_sms = 0;
    // options
    int basis = 0, spmv_variant = 0, lanes_opt = 0, use_graph = 1, spmv_depth = 2, block_variant = 0, form = 0, resident_opt = 0, reorder_opt = 0, replace_every = 0, method = 0, pdl = 1;
    // problem (borrowed CSR)
    int64_t n = 0, nnz = 0;
    int s = 0;
    const int* rp = nullptr;
    const int* ci = nullptr;
    const double* va = nullptr;
    const double* b_cur = nullptr;  // right-hand side of the solve in progress (solver's numbering), for residual replacement
    bool ready = false, in_solve = false;
    // owned device memory
    double *dinv = nullptr, *R = nullptr, *AR = nullptr, *P = nullptr, *AP = nullptr, *x = nullptr, *r = nullptr;
    double* partials = nullptr;
    double* mom = nullptr;        // moment form: [2s][spmv_grid] per-block partials of mu^1 .. mu^{2s-1}
    ScgState* st = nullptr;       // production state
    ScgState* st_test = nullptr;  // state used by the test hooks
    int* iscratch = nullptr;      // [err, max_len, max_tile]
    // owned copies made by solve_host
    int *own_rp = nullptr, *own_ci = nullptr;
    int64_t own_n = 0, own_nnz = 0;  // sizes the owned copies were allocated for (solve_host reuses them call to call)
    double *own_va = nullptr, *own_b = nullptr, *own_x = nullptr;
    // kernel configuration
    int lanes = 1;
    bool bulk = false;
    int bulk_cap = 256, bulk_wpc = 8;
    bool cta = false;             // thread-per-row matrices: CTA-pipelined SpMV (spmv_cta.cuh) instead of the per-warp rings
    int cta_depth = 2, cta_minb = 3, cta_tiles = 0;
    bool cta2_small = false;      // two lanes per row: the 96-row / three-CTA shape (Gram-form handles)
    int spmv_grid = 0, gram_grid = 0, update_grid = 0, init_grid = 0, pcg_grid = 0;
    bool staged = false;       // update through the TMA tile pipeline (s >= 5)
    bool staged_gram = false;  // Gram through the TMA tile pipeline (every s: see gram_tma.cuh)
    int gram_grid_reg = 0, update_grid_reg = 0;  // grids of the register kernels (used by hooks on misaligned buffers)
    int gram_tile = 0, gram_depth = 0, update_tile = 0, update_depth = 0;  // staged kernels: rows per tile, ring slots (0 = not staged)
    int64_t num_tiles = 0;
    int max_row_len = 0;
    double dinv_uniform = 0.0;  // 1 / a_ii if the diagonal is constant (then the update kernels skip the dinv stream), else 0
    // locality reordering (reorder.cuh): A' = Pi A Pi^T in owned arrays; rp/ci/va above then point at them
    bool reordered = false;
    int *perm = nullptr, *rank = nullptr;        // perm[new] = old, rank[old] = new
    int *own_prp = nullptr, *own_pci = nullptr;
    double *own_pva = nullptr, *bperm = nullptr, *x0perm = nullptr;
    int cm_levels = 0, cm_comps = 0, far_permille = 0;
    // resident (cooperative, whole loop in one launch) path for problems that fit shared memory
    bool resident = false;
    int resident_sync = 0;               // 0 = flag-in-data exchange between the CTAs (default) | 1 = grid barriers (round 1)
    ulonglong2 *llR = nullptr, *llPart = nullptr, *llTot = nullptr;  // tagged exchange buffers of the resident kernel
    size_t llR_bytes = 0, llPart_bytes = 0;  // (llTot has the size of llPart)
    unsigned int ll_tag = 0;             // tags below or equal to this value have been used
    int res_grid = 0, res_rpb = 0, res_nzcap = 0, res_threads = 0;
    size_t res_smem = 0;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t gexec = nullptr;
    // host polling
    Header* h_hdr = nullptr;  // pinned, 2 entries
    cudaEvent_t ev[2] = {nullptr, nullptr};
    // bookkeeping
    int64_t launches = 0;
    int64_t graph_launches = 0;
    double rtol = 0.0;
    std::chrono::steady_clock::time_point t_begin;
    std::string err;
};

namespace {

int fail(sstep_cg* h, int code, const std::string& msg) {
    if (h) h->err = msg;
    return code;
}

#define CK(call)                                                                                              \
    do {                                                                                                      \
        cudaError_t e_ = (call);                                                                              \
        if (e_ != cudaSuccess)                                                                                \
            return fail(h, SSTEP_CG_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_));            \
    } while (0)

// ---------------------------------------------------------------- kernel dispatch
using bulk_fn_t = void (*)(int, int, const int*, const int*, const double*, const double*, double*, double*,
                           const double*, int, const ScgState*, int, double*, double*);

// launch of a hot-path kernel (every one of them starts with pdl_wait, common.cuh): with option pdl the launch carries
// the programmatic-stream-serialization attribute, which stream capture turns into programmatic edges of the graph
template <typename... Exp, typename... Act>
cudaError_t launch_k(const sstep_cg* h, void (*kern)(Exp...), unsigned grid, unsigned block, size_t smem, cudaStream_t sm,
                     Act&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = sm;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = h->pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<Exp>(args)...);
}

template <int L, bool MOM>
bulk_fn_t bulk_kernel_mom(int depth) {
    switch (depth) {
        case 2: return spmv_bulk_kernel<L, 2, BULK_CAP, BULK_WPC, MOM>;
        case 3: return spmv_bulk_kernel<L, 3, BULK_CAP, BULK_WPC, MOM>;
        default: return spmv_bulk_kernel<L, 4, BULK_CAP, BULK_WPC, MOM>;
    }
}
template <int L>
bulk_fn_t bulk_kernel_for(int depth, bool mom, int cap) {
    if constexpr (L == 1) {
        if (cap == BULK_CAP1) return mom ? spmv_bulk_kernel<1, 2, BULK_CAP1, BULK_WPC1, true, 2> : spmv_bulk_kernel<1, 2, BULK_CAP1, BULK_WPC1, false, 2>;
    }
    if constexpr (L == 2) {
        if (cap == BULK_CAP2) return mom ? spmv_bulk_kernel<2, 2, BULK_CAP2, BULK_WPC2, true, 2> : spmv_bulk_kernel<2, 2, BULK_CAP2, BULK_WPC2, false, 2>;
        if (cap == BULK_CAP2B) return mom ? spmv_bulk_kernel<2, 2, BULK_CAP2B, BULK_WPC2B, true, 2> : spmv_bulk_kernel<2, 2, BULK_CAP2B, BULK_WPC2B, false, 2>;
    }
    return mom ? bulk_kernel_mom<L, true>(depth) : bulk_kernel_mom<L, false>(depth);
}

using cta_fn_t = void (*)(int, int, const int*, const int*, const double*, const double*, double*, double*,
                          const double*, int, const ScgState*, int, double*, double*, double);
template <bool MOM, bool UNI>
cta_fn_t cta_kernel_mu(int depth, int minb) {
    if (minb == 2) {
        switch (depth) {
            case 2: return spmv_cta_kernel<2, CTA_TR, CTA_CAPT, MOM, 2, UNI>;
            case 3: return spmv_cta_kernel<3, CTA_TR, CTA_CAPT, MOM, 2, UNI>;
            default: return spmv_cta_kernel<4, CTA_TR, CTA_CAPT, MOM, 2, UNI>;
        }
    }
    switch (depth) {
        case 2: return spmv_cta_kernel<2, CTA_TR, CTA_CAPT, MOM, 3, UNI>;
        case 3: return spmv_cta_kernel<3, CTA_TR, CTA_CAPT, MOM, 3, UNI>;
        default: return spmv_cta_kernel<4, CTA_TR, CTA_CAPT, MOM, 3, UNI>;
    }
}
cta_fn_t cta_kernel_for(const sstep_cg* h, bool mom) {
    const bool uni = h->dinv_uniform > 0.0;
    if (h->lanes == 2) {
        if (h->cta2_small)  // Gram-form handles only: never launched with moment partials
            return uni ? spmv_cta_kernel<2, CTA2B_TR, CTA2B_CAPT, false, 3, true, 2, CTA2_U> : spmv_cta_kernel<2, CTA2B_TR, CTA2B_CAPT, false, 3, false, 2, CTA2_U>;
        if (mom) return uni ? spmv_cta_kernel<2, CTA2_TR, CTA2_CAPT, true, 2, true, 2, CTA2_U> : spmv_cta_kernel<2, CTA2_TR, CTA2_CAPT, true, 2, false, 2, CTA2_U>;
        return uni ? spmv_cta_kernel<2, CTA2_TR, CTA2_CAPT, false, 2, true, 2, CTA2_U> : spmv_cta_kernel<2, CTA2_TR, CTA2_CAPT, false, 2, false, 2, CTA2_U>;
    }
    if (mom) return uni ? cta_kernel_mu<true, true>(h->cta_depth, h->cta_minb) : cta_kernel_mu<true, false>(h->cta_depth, h->cta_minb);
    return uni ? cta_kernel_mu<false, true>(h->cta_depth, h->cta_minb) : cta_kernel_mu<false, false>(h->cta_depth, h->cta_minb);
}
size_t cta_smem_for(const sstep_cg* h) {
    const int depth = h->lanes == 2 ? 2 : h->cta_depth, capt = h->lanes == 2 ? (h->cta2_small ? CTA2B_CAPT : CTA2_CAPT) : CTA_CAPT;
    return (size_t)depth * capt * 12 + (size_t)depth * 24;
}
int cta_threads(const sstep_cg* h) { return (h->lanes == 2 ? 2 * (h->cta2_small ? CTA2B_TR : CTA2_TR) : CTA_TR) + 32; }  // consumer warps + the producer warp
int cta_per_sm(const sstep_cg* h) { return h->lanes == 2 ? (h->cta2_small ? 3 : 2) : h->cta_minb; }

template <int L>
cudaError_t launch_spmv_L(sstep_cg* h, cudaStream_t sm, const double* x, double* y, double* yjac, const double* xprev,
                          int mode, const ScgState* st, double* mom_a, double* mom_b) {
    if ((L == 1 || L == 2) && h->cta) {
        return launch_k(h, cta_kernel_for(h, mom_a != nullptr), h->spmv_grid, cta_threads(h), cta_smem_for(h), sm, (int)h->n,
                        (int)h->nnz, h->rp, h->ci, h->va, x, y, yjac, xprev, mode, st, h->cta_tiles, mom_a, mom_b, h->dinv_uniform);
    }
    if (h->bulk) {
        return launch_k(h, bulk_kernel_for<L>(h->spmv_depth, mom_a != nullptr, h->bulk_cap), h->spmv_grid, h->bulk_wpc * 32,
                        bulk_smem_for(h->spmv_depth, h->bulk_cap, h->bulk_wpc), sm, (int)h->n, (int)h->nnz, h->rp, h->ci, h->va,
                        x, y, yjac, xprev, mode, st, (int)h->num_tiles, mom_a, mom_b);
    }
    if (mom_a) return launch_k(h, spmv_vec_kernel<L, true>, h->spmv_grid, 256, 0, sm, h->n, h->rp, h->ci, h->va, h->dinv, x, y, yjac, xprev, mode, st, mom_a, mom_b);
    return launch_k(h, spmv_vec_kernel<L, false>, h->spmv_grid, 256, 0, sm, h->n, h->rp, h->ci, h->va, h->dinv, x, y, yjac, xprev, mode, st, mom_a, mom_b);
}

cudaError_t launch_spmv(sstep_cg* h, cudaStream_t sm, const double* x, double* y, double* yjac, const double* xprev,
                        int mode, const ScgState* st, double* mom_a = nullptr, double* mom_b = nullptr) {
    h->launches++;
    switch (h->lanes) {
        case 1: return launch_spmv_L<1>(h, sm, x, y, yjac, xprev, mode, st, mom_a, mom_b);
        case 2: return launch_spmv_L<2>(h, sm, x, y, yjac, xprev, mode, st, mom_a, mom_b);
        case 4: return launch_spmv_L<4>(h, sm, x, y, yjac, xprev, mode, st, mom_a, mom_b);
        case 8: return launch_spmv_L<8>(h, sm, x, y, yjac, xprev, mode, st, mom_a, mom_b);
        case 16: return launch_spmv_L<16>(h, sm, x, y, yjac, xprev, mode, st, mom_a, mom_b);
        default: return launch_spmv_L<32>(h, sm, x, y, yjac, xprev, mode, st, mom_a, mom_b);
    }
}

template <int L>
cudaError_t config_spmv_L(sstep_cg* h) {
    int occ = 0;
    cudaError_t e;
    if ((L == 1 || L == 2) && h->cta) {
        const size_t smem = cta_smem_for(h);
        for (int mom = 0; mom < 2; mom++) {
            e = cudaFuncSetAttribute(cta_kernel_for(h, mom != 0), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
        }
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, cta_kernel_for(h, h->form != 0 || h->method == 1), cta_threads(h), smem);
        if (e != cudaSuccess) return e;
        if (occ < 1) occ = 1;
        if (occ > cta_per_sm(h)) occ = cta_per_sm(h);
        const int64_t cap = (int64_t)occ * h->num_sms;
        h->spmv_grid = (int)(h->cta_tiles < cap ? h->cta_tiles : cap);
        if (h->spmv_grid < 1) h->spmv_grid = 1;
        return cudaSuccess;
    }
    if (h->bulk) {
        auto k = bulk_kernel_for<L>(h->spmv_depth, h->form != 0 || h->method == 1, h->bulk_cap);
        const size_t smem = bulk_smem_for(h->spmv_depth, h->bulk_cap, h->bulk_wpc);
        e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        // (the variant without moments is also launched in the moment form: x0 != 0 start-up, test_spmv hook)
        e = cudaFuncSetAttribute(bulk_kernel_for<L>(h->spmv_depth, false, h->bulk_cap), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, h->bulk_wpc * 32, smem);
        if (e != cudaSuccess) return e;
        if (occ < 1) occ = 1;
        int64_t want = (h->num_tiles + h->bulk_wpc - 1) / h->bulk_wpc;
        int64_t cap = (int64_t)occ * h->num_sms;
        h->spmv_grid = (int)(want < cap ? want : cap);
    } else {
        auto k = spmv_vec_kernel<L, false>;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, 256, 0);
        if (e != cudaSuccess) return e;
        if (occ < 1) occ = 1;
        int64_t rows_per_block = 256 / L;
        int64_t want = (h->n + rows_per_block - 1) / rows_per_block;
        int64_t cap = (int64_t)occ * h->num_sms * 4;
        h->spmv_grid = (int)(want < cap ? want : cap);
    }
    if (h->spmv_grid < 1) h->spmv_grid = 1;
    return cudaSuccess;
}

cudaError_t config_spmv(sstep_cg* h) {
    switch (h->lanes) {
        case 1: return config_spmv_L<1>(h);
        case 2: return config_spmv_L<2>(h);
        case 4: return config_spmv_L<4>(h);
        case 8: return config_spmv_L<8>(h);
        case 16: return config_spmv_L<16>(h);
        default: return config_spmv_L<32>(h);
    }
}

inline bool aligned16(const void* p) { return ((uintptr_t)p & 15) == 0; }

template <int S>
cudaError_t gram_S(sstep_cg* h, cudaStream_t sm, bool configure, const double* R, const double* AR, const double* AP,
                   const double* r, ScgState* st, int do_solve) {
    using Cfg = GramCfg<S>;
    using TC = GramTmaCfg<S>;
    if (configure) {
        int occ = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, gram_kernel<S>, Cfg::NW * 32, 0);
        if (e != cudaSuccess) return e;
        if (occ < 1) occ = 1;
        int64_t want = (h->n + Cfg::RG * 32 - 1) / (Cfg::RG * 32);
        int64_t cap = (int64_t)occ * h->num_sms;
        h->gram_grid_reg = h->gram_grid = (int)(want < cap ? want : cap);
        if (h->staged_gram) {
            e = cudaFuncSetAttribute(gram_tma_kernel<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC::SMEM);
            if (e != cudaSuccess) return e;
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, gram_tma_kernel<S>, TC::THREADS, TC::SMEM);
            if (e != cudaSuccess) return e;
            if (occ < 1) occ = 1;
            want = (h->n + TC::T - 1) / TC::T;
            cap = (int64_t)occ * h->num_sms;
            h->gram_grid = (int)(want < cap ? want : cap);
            if (h->gram_grid < h->gram_grid_reg) h->gram_grid_reg = h->gram_grid;  // partials are sized by gram_grid
        }
        h->gram_tile = h->staged_gram ? TC::T : 0;
        h->gram_depth = h->staged_gram ? TC::D : 0;
        return cudaSuccess;
    }
    if (h->staged_gram && aligned16(R) && aligned16(AR) && aligned16(AP) && aligned16(r)) {
        return launch_k(h, gram_tma_kernel<S>, h->gram_grid, TC::THREADS, TC::SMEM, sm, h->n, R, AR, AP, r, h->partials, st, do_solve,
                        (h->n + TC::T - 1) / TC::T);
    }
    return launch_k(h, gram_kernel<S>, h->gram_grid_reg, Cfg::NW * 32, 0, sm, h->n, R, AR, AP, r, h->partials, st, do_solve);
}

template <int S, bool MOM>
cudaError_t update_SM(sstep_cg* h, cudaStream_t sm, bool configure, double* R, const double* AR, double* P, double* AP,
                      double* x, double* r, const double* beta, const double* alpha, ScgState* st, double* rho_out) {
    using TC = UpdateTmaCfg<S>;
    if (configure) {
        int occ = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, update_kernel<S, MOM>, 256, 0);
        if (e != cudaSuccess) return e;
        if (occ < 1) occ = 1;
        int64_t want = (h->n + 255) / 256;
        int64_t cap = (int64_t)occ * h->num_sms;
        h->update_grid_reg = h->update_grid = (int)(want < cap ? want : cap);
        if (h->staged) {
            e = cudaFuncSetAttribute(update_tma_kernel<S, MOM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC::SMEM);
            if (e != cudaSuccess) return e;
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, update_tma_kernel<S, MOM>, TC::THREADS, TC::SMEM);
            if (e != cudaSuccess) return e;
            if (occ < 1) occ = 1;
            want = (h->n + TC::T - 1) / TC::T;
            cap = (int64_t)occ * h->num_sms;
            h->update_grid = (int)(want < cap ? want : cap);
            if (h->update_grid < h->update_grid_reg) h->update_grid_reg = h->update_grid;
        }
        h->update_tile = h->staged ? TC::T : 0;
        h->update_depth = h->staged ? TC::D : 0;
        return cudaSuccess;
    }
    if (h->staged && aligned16(R) && aligned16(AR) && aligned16(P) && aligned16(AP) && aligned16(x) && aligned16(r)) {
        return launch_k(h, update_tma_kernel<S, MOM>, h->update_grid, TC::THREADS, TC::SMEM, sm, h->n, R, AR, P, AP, x, r, h->dinv,
                        beta, alpha, h->partials, st, rho_out, (h->n + TC::T - 1) / TC::T);
    }
    if constexpr (S == 1) {  // two rows per thread, 128-bit accesses (update.cuh); the grid of update_kernel<1> covers it
        if (aligned16(R) && aligned16(AR) && aligned16(P) && aligned16(AP) && aligned16(x) && aligned16(r) && aligned16(h->dinv))
            return launch_k(h, update1_kernel<MOM>, h->update_grid_reg, 256, 0, sm, h->n, R, AR, P, AP, x, r, h->dinv, beta, alpha,
                            h->partials, st, rho_out, h->dinv_uniform);
    }
    return launch_k(h, update_kernel<S, MOM>, h->update_grid_reg, 256, 0, sm, h->n, R, AR, P, AP, x, r, h->dinv, beta, alpha,
                    h->partials, st, rho_out, h->dinv_uniform);
}

// the moment form's update also accumulates mu^0 = R_1^T r (compiled in only there)
template <int S>
cudaError_t update_S(sstep_cg* h, cudaStream_t sm, bool configure, double* R, const double* AR, double* P, double* AP,
                     double* x, double* r, const double* beta, const double* alpha, ScgState* st, double* rho_out) {
    return h->form ? update_SM<S, true>(h, sm, configure, R, AR, P, AP, x, r, beta, alpha, st, rho_out)
                   : update_SM<S, false>(h, sm, configure, R, AR, P, AP, x, r, beta, alpha, st, rho_out);
}

#define SCG_DISPATCH_S(fn, ...)                          \
    switch (h->s) {                                      \
        case 1: return fn<1>(__VA_ARGS__);               \
        case 2: return fn<2>(__VA_ARGS__);               \
        case 3: return fn<3>(__VA_ARGS__);               \
        case 4: return fn<4>(__VA_ARGS__);               \
        case 5: return fn<5>(__VA_ARGS__);               \
        case 6: return fn<6>(__VA_ARGS__);               \
        case 7: return fn<7>(__VA_ARGS__);               \
        case 8: return fn<8>(__VA_ARGS__);               \
        case 9: return fn<9>(__VA_ARGS__);               \
        case 10: return fn<10>(__VA_ARGS__);             \
        case 11: return fn<11>(__VA_ARGS__);             \
        case 12: return fn<12>(__VA_ARGS__);             \
        case 13: return fn<13>(__VA_ARGS__);             \
        case 14: return fn<14>(__VA_ARGS__);             \
        case 15: return fn<15>(__VA_ARGS__);             \
        default: return fn<16>(__VA_ARGS__);             \
    }

cudaError_t launch_gram(sstep_cg* h, cudaStream_t sm, bool configure, const double* R, const double* AR, const double* AP,
                        const double* r, ScgState* st, int do_solve) {
    if (!configure) h->launches++;
    SCG_DISPATCH_S(gram_S, h, sm, configure, R, AR, AP, r, st, do_solve)
}

cudaError_t launch_update(sstep_cg* h, cudaStream_t sm, bool configure, double* R, const double* AR, double* P, double* AP,
                          double* x, double* r, const double* beta, const double* alpha, ScgState* st, double* rho_out) {
    if (!configure) h->launches++;
    SCG_DISPATCH_S(update_S, h, sm, configure, R, AR, P, AP, x, r, beta, alpha, st, rho_out)
}

// resident path (resident.cuh): op 0 = set the shared-memory attribute and report the occupancy, op 1 = cooperative launch
template <int S, bool LL>
cudaError_t resident_SL(sstep_cg* h, cudaStream_t sm, int op, int kmax, int* occ_out) {
    if (op == 0) {
        cudaError_t e = cudaFuncSetAttribute(resident_kernel<S, LL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->res_smem);
        if (e != cudaSuccess) return e;
        return cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ_out, resident_kernel<S, LL>, h->res_threads, h->res_smem);
    }
    ResidentParams p;
    p.n = (int)h->n; p.rpb = h->res_rpb; p.nzcap = h->res_nzcap; p.kmax = kmax; p.basis = h->basis;
    p.rp = h->rp; p.ci = h->ci; p.va = h->va; p.dinv = h->dinv;
    p.Rg = h->R; p.ARg = h->AR; p.P = h->P; p.AP = h->AP; p.x = h->x; p.r = h->r;
    p.partials = h->partials; p.st = h->st;
    p.llR = h->llR; p.llPart = h->llPart; p.llTot = h->llTot; p.tag0 = h->ll_tag;
    void* args[] = {&p};
    return cudaLaunchCooperativeKernel((const void*)resident_kernel<S, LL>, dim3(h->res_grid), dim3(h->res_threads), args, h->res_smem, sm);
}
template <int S>
cudaError_t resident_S(sstep_cg* h, cudaStream_t sm, int op, int kmax, int* occ_out) {
    return h->resident_sync == 0 ? resident_SL<S, true>(h, sm, op, kmax, occ_out) : resident_SL<S, false>(h, sm, op, kmax, occ_out);
}

cudaError_t resident_op(sstep_cg* h, cudaStream_t sm, int op, int kmax, int* occ_out) {
    SCG_DISPATCH_S(resident_S, h, sm, op, kmax, occ_out)
}

// Alg. 4 on the given buffers: s Jacobi-fused SpMVs (R(:,1) must already hold D^-1 r)
cudaError_t launch_mpk(sstep_cg* h, cudaStream_t sm, double* R, double* AR, const ScgState* st) {
    const int64_t n = h->n;
    for (int j = 0; j < h->s; j++) {
        double* yjac = (j + 1 < h->s) ? R + (int64_t)(j + 1) * n : nullptr;
        int mode = 0;
        const double* xprev = nullptr;
        if (h->basis == SSTEP_CG_BASIS_CHEBYSHEV) {
            mode = (j == 0) ? 1 : 2;
            if (j > 0) xprev = R + (int64_t)(j - 1) * n;
        }
        // moment form: SpMV j (1-based) also leaves the per-block partials of mu^{2j-1} = R_j^T AR_j and mu^{2j} = R_{j+1}^T AR_j
        double* mom_a = h->form ? h->mom + (int64_t)(2 * j + 1) * h->spmv_grid : nullptr;
        double* mom_b = (h->form && j + 1 < h->s) ? h->mom + (int64_t)(2 * j + 2) * h->spmv_grid : nullptr;
        cudaError_t e = launch_spmv(h, sm, R + (int64_t)j * n, AR + (int64_t)j * n, yjac, xprev, mode, st, mom_a, mom_b);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// moment form, after the MPK: fixed-order sum of the moment partials + Alg. 6 in one warp (replaces the Gram kernel)
cudaError_t launch_sw(sstep_cg* h, cudaStream_t sm, ScgState* st, int do_solve) {
    h->launches++;
    return launch_k(h, sw_kernel, 1, 256, 0, sm, h->s, h->spmv_grid, h->mom, st, do_solve);
}

// one iteration of Alg. 1 (method = 1; pcg.cuh): p = P, s_k = AP, u = R
cudaError_t launch_pcg_iteration(sstep_cg* h, cudaStream_t sm, cudaEvent_t* evs = nullptr) {
    if (evs) cudaEventRecord(evs[0], sm);
    cudaError_t e = launch_spmv(h, sm, h->P, h->AP, nullptr, nullptr, 0, h->st, h->mom, nullptr);
    if (e != cudaSuccess) return e;
    if (evs) { cudaEventRecord(evs[1], sm); cudaEventRecord(evs[2], sm); }
    pcg_update_kernel<<<h->pcg_grid, 256, 0, sm>>>(h->n, h->P, h->AP, h->x, h->r, h->R, h->dinv, h->mom, h->spmv_grid,
                                                         h->partials, h->st, h->dinv_uniform);
    if (evs) { cudaEventRecord(evs[3], sm); cudaEventRecord(evs[4], sm); }
    pcg_direction_kernel<<<h->pcg_grid, 256, 0, sm>>>(h->n, h->R, h->P, h->st);
    if (evs) cudaEventRecord(evs[5], sm);
    h->launches += 2;
    return cudaGetLastError();
}

// one outer iteration on the production buffers (Alg. 3 l.5-21)
cudaError_t launch_outer(sstep_cg* h, cudaStream_t sm) {
    if (h->method == 1) return launch_pcg_iteration(h, sm);
    cudaError_t e = launch_mpk(h, sm, h->R, h->AR, h->st);
    if (e != cudaSuccess) return e;
    e = h->form ? launch_sw(h, sm, h->st, 1) : launch_gram(h, sm, false, h->R, h->AR, h->AP, h->r, h->st, 1);
    if (e != cudaSuccess) return e;
    return launch_update(h, sm, false, h->R, h->AR, h->P, h->AP, h->x, h->r, h->st->beta, h->st->alpha, h->st, nullptr);
}

void free_problem(sstep_cg* h) {
    if (h->gexec) cudaGraphExecDestroy(h->gexec);
    if (h->graph) cudaGraphDestroy(h->graph);
    h->gexec = nullptr;
    h->graph = nullptr;
    double** bufs[] = {&h->dinv, &h->R, &h->AR, &h->P, &h->AP, &h->x, &h->r, &h->partials, &h->mom};
    for (double** b : bufs) {
        if (*b) cudaFree(*b);
        *b = nullptr;
    }
    int** ibufs[] = {&h->perm, &h->rank, &h->own_prp, &h->own_pci};
    for (int** b : ibufs) {
        if (*b) cudaFree(*b);
        *b = nullptr;
    }
    if (h->llR) cudaFree(h->llR);
    if (h->llPart) cudaFree(h->llPart);
    if (h->llTot) cudaFree(h->llTot);
    h->llR = h->llPart = h->llTot = nullptr;
    double** dbufs[] = {&h->own_pva, &h->bperm, &h->x0perm};
    for (double** b : dbufs) {
        if (*b) cudaFree(*b);
        *b = nullptr;
    }
    h->reordered = false;
    h->ready = false;
    h->in_solve = false;
}

void free_owned(sstep_cg* h) {
    if (h->own_rp) cudaFree(h->own_rp);
    if (h->own_ci) cudaFree(h->own_ci);
    if (h->own_va) cudaFree(h->own_va);
    if (h->own_b) cudaFree(h->own_b);
    if (h->own_x) cudaFree(h->own_x);
    h->own_rp = h->own_ci = nullptr;
    h->own_va = h->own_b = h->own_x = nullptr;
    h->own_n = h->own_nnz = 0;
}

int kernels_per_outer(const sstep_cg* h) {
    if (h->method == 1) return 3;
    return h->s + 2;
}

__global__ void iota_kernel(int64_t n, int* __restrict__ p) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = (int)i;
}

// ---------------------------------------------------------------- the steps of sstep_cg_setup (each returns 0 or an error code)
// validation of the CSR arrays, dinv = 1 / a_ii, longest row
int setup_analyze(sstep_cg* h) {
    const int64_t n = h->n;
    const int64_t nnz = h->nnz;
    cudaStream_t sm = h->stream;
    const int* rowptr = h->rp;
    const int* colidx = h->ci;
    const double* vals = h->va;
    int hs[4] = {0, 0, 0, 0};
    CK(cudaMalloc(&h->dinv, sizeof(double) * n));
    CK(cudaMemsetAsync(h->iscratch, 0, 4 * sizeof(int), sm));
    analyze_kernel<<<(unsigned)((n + 255) / 256), 256, 0, sm>>>(n, nnz, rowptr, colidx, vals, h->dinv, h->iscratch, h->iscratch + 1);
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(hs, h->iscratch, 2 * sizeof(int), cudaMemcpyDeviceToHost, sm));
    CK(cudaStreamSynchronize(sm));
    if (hs[0]) {
        char buf[160];
        snprintf(buf, sizeof buf, "setup: invalid matrix (flags %d: 1 rowptr, 2 column index, 4 diagonal missing, duplicated or <= 0)", hs[0]);
        free_problem(h);
        return fail(h, SSTEP_CG_ERR_MATRIX, buf);
    }
    h->max_row_len = hs[1];
    return 0;
}

// locality test and, if wanted, the Cuthill-McKee renumbering (h->rp / ci / va then point at the owned permuted copy)
int setup_reorder(sstep_cg* h) {
    const int64_t n = h->n;
    const int64_t nnz = h->nnz;
    cudaStream_t sm = h->stream;
    const int* rowptr = h->rp;
    const int* colidx = h->ci;
    const double* vals = h->va;
    int hs[4] = {0, 0, 0, 0};
    // auto: only when the gathered vector cannot live in L2 (n >= 2^23 rows = 67 MB) and more than a quarter of the
    // entries reach further than 2^20 rows (8 MB) from the diagonal
    {
        unsigned long long* far = nullptr;
        unsigned long long hfar = 0;
        CK(cudaMalloc(&far, sizeof(unsigned long long)));
        CK(cudaMemsetAsync(far, 0, sizeof(unsigned long long), sm));
        scg_reorder::far_entries_kernel<<<(unsigned)((n + 255) / 256), 256, 0, sm>>>(n, rowptr, colidx, 1 << 20, far);
        CK(cudaMemcpyAsync(&hfar, far, sizeof(unsigned long long), cudaMemcpyDeviceToHost, sm));
        CK(cudaStreamSynchronize(sm));
        cudaFree(far);
        h->far_permille = (int)(1000.0 * (double)hfar / (double)nnz);
    }
    h->cm_levels = h->cm_comps = 0;
    if (h->reorder_opt == 2 || (h->reorder_opt == 0 && n >= (int64_t(1) << 23) && h->far_permille > 250)) {
        CK(cudaMalloc(&h->perm, sizeof(int) * (size_t)n));
        CK(cudaMalloc(&h->rank, sizeof(int) * (size_t)n));
        bool done = false;
        CK(scg_reorder::cuthill_mckee((int)n, rowptr, colidx, sm, h->perm, h->rank, &done, &h->cm_levels, &h->cm_comps));
        if (done) {
            CK(cudaMalloc(&h->own_prp, sizeof(int) * ((size_t)n + 1)));
            CK(cudaMalloc(&h->own_pci, sizeof(int) * (size_t)nnz));
            CK(cudaMalloc(&h->own_pva, sizeof(double) * (size_t)nnz));
            CK(cudaMalloc(&h->bperm, sizeof(double) * (size_t)n));
            CK(cudaMalloc(&h->x0perm, sizeof(double) * (size_t)n));
            CK(scg_reorder::permute_csr((int)n, (int)nnz, h->perm, h->rank, rowptr, colidx, vals, h->own_prp, h->own_pci, h->own_pva, sm));
            h->rp = rowptr = h->own_prp;
            h->ci = colidx = h->own_pci;
            h->va = vals = h->own_pva;
            h->reordered = true;
            // dinv and the row statistics of the permuted matrix (same validation, now of our own copy)
            CK(cudaMemsetAsync(h->iscratch, 0, 4 * sizeof(int), sm));
            analyze_kernel<<<(unsigned)((n + 255) / 256), 256, 0, sm>>>(n, nnz, rowptr, colidx, vals, h->dinv, h->iscratch, h->iscratch + 1);
            CK(cudaGetLastError());
            CK(cudaMemcpyAsync(hs, h->iscratch, 2 * sizeof(int), cudaMemcpyDeviceToHost, sm));
            CK(cudaStreamSynchronize(sm));
            if (hs[0]) {
                free_problem(h);
                return fail(h, SSTEP_CG_ERR_CUDA, "setup: internal error, the permuted matrix failed validation");
            }
        } else {
            cudaFree(h->perm); cudaFree(h->rank);
            h->perm = h->rank = nullptr;
        }
    }
    return 0;
}

// is the diagonal constant?
int setup_uniform_diagonal(sstep_cg* h) {
    const int64_t n = h->n;
    cudaStream_t sm = h->stream;
    {
        int one = 1, flag = 0;
        double d0 = 0.0;
        CK(cudaMemcpyAsync(h->iscratch + 3, &one, sizeof(int), cudaMemcpyHostToDevice, sm));
        uniform_diag_kernel<<<(unsigned)((n + 255) / 256), 256, 0, sm>>>(n, h->dinv, h->iscratch + 3);
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(&flag, h->iscratch + 3, sizeof(int), cudaMemcpyDeviceToHost, sm));
        CK(cudaMemcpyAsync(&d0, h->dinv, sizeof(double), cudaMemcpyDeviceToHost, sm));
        CK(cudaStreamSynchronize(sm));
        h->dinv_uniform = (flag == 1 && d0 > 0.0) ? d0 : 0.0;
    }
    return 0;
}

// lanes per row and generic / bulk-staged SpMV (tile shape) from the row statistics
int setup_spmv_variant(sstep_cg* h) {
    const int64_t n = h->n;
    const int64_t nnz = h->nnz;
    cudaStream_t sm = h->stream;
    const int* rowptr = h->rp;
    const int* colidx = h->ci;
    const double* vals = h->va;
    int hs[4] = {0, 0, 0, 0};
    const double mean = (double)nnz / (double)n;
    int L = 1;
    while (L < 32 && mean / L > 8.0) L *= 2;
    if (h->lanes_opt) L = h->lanes_opt;
    h->bulk = false;
    const bool aligned = (((uintptr_t)colidx | (uintptr_t)vals) & 15) == 0;
    // auto: the bulk-staged kernel for thread-per-row matrices (mean row <= 8 entries, e.g. 7-point stencils), where it
    // reaches the copy peak, and -- with TWO lanes per row and 512-entry tiles -- for mean rows of 16..32 entries
    // (27-point 160^3: 257 us against 272 us for the generic kernel at L = 4 and 285 us for bulk tiles at L = 4: few lanes
    // per row keep the x gathers of a warp on consecutive addresses).  Forced (spmv_variant = 2): any L whose tiles fit.
    const bool auto_bulk = h->spmv_variant == 0 && (L == 1 || (L == 4 && !h->lanes_opt && h->spmv_depth == 2));
    if ((h->spmv_variant == 2 || auto_bulk) && aligned && n + 64 < (int64_t(1) << 31)) {
        if (auto_bulk && L == 4) L = 2;
        for (int Lb = L; Lb <= 32; Lb *= 2) {
            const int rpt = 32 / Lb;
            const int64_t tiles = (n + rpt - 1) / rpt;
            CK(cudaMemsetAsync(h->iscratch + 2, 0, sizeof(int), sm));
            tile_nnz_max_kernel<<<(unsigned)((tiles + 255) / 256), 256, 0, sm>>>(n, rowptr, rpt, tiles, h->iscratch + 2);
            CK(cudaGetLastError());
            CK(cudaMemcpyAsync(hs + 2, h->iscratch + 2, sizeof(int), cudaMemcpyDeviceToHost, sm));
            CK(cudaStreamSynchronize(sm));
            int cap = 0, wpc = BULK_WPC;
            if (hs[2] + 3 <= BULK_CAP) cap = BULK_CAP;
            else if (Lb == 2 && h->spmv_depth == 2 && hs[2] + 3 <= BULK_CAP2) { cap = BULK_CAP2; wpc = BULK_WPC2; }
            else if (Lb == 2 && h->spmv_depth == 2 && hs[2] + 3 <= BULK_CAP2B) { cap = BULK_CAP2B; wpc = BULK_WPC2B; }
            else if (Lb == 1 && h->spmv_variant == 2 && h->spmv_depth == 2 && hs[2] + 3 <= BULK_CAP1) { cap = BULK_CAP1; wpc = BULK_WPC1; }
            if (cap) {
                h->bulk = true;
                h->bulk_cap = cap;
                h->bulk_wpc = wpc;
                L = Lb;
                h->num_tiles = tiles;
                break;
            }
            if (h->lanes_opt || h->spmv_variant == 0) break;
        }
        if (auto_bulk && !h->bulk && L == 2) L = 4;  // tiles too large: back to the generic kernel at its own L
    }
    if (h->spmv_variant == 2 && !h->bulk) {
        free_problem(h);
        return fail(h, SSTEP_CG_ERR_ARG, "setup: bulk SpMV forced but a tile exceeds the staging capacity or arrays are not 16 B aligned");
    }
    // thread-per-row matrices whose 256-row tiles fit a stage: the CTA-pipelined kernel (few large bulk copies in flight,
    // spmv_cta.cuh) replaces the per-warp rings -- auto, or forced with spmv_variant = 3 (2 keeps the per-warp rings)
    h->cta = false;
    if (h->spmv_variant == 3 && L == 4 && !h->lanes_opt) L = 2;  // (forced: the two-lane shape for mean rows of 16-32 entries)
    if (((h->spmv_variant == 0 && h->bulk) || h->spmv_variant == 3) && (L == 1 || L == 2) && aligned &&
        n + 2 * CTA_TR < (int64_t(1) << 31)) {
        h->cta2_small = (L == 2) && h->form == 0 && h->method == 0;
        const int tr = (L == 2) ? (h->cta2_small ? CTA2B_TR : CTA2_TR) : CTA_TR, capt = (L == 2) ? (h->cta2_small ? CTA2B_CAPT : CTA2_CAPT) : CTA_CAPT;
        const int64_t tiles = (n + tr - 1) / tr;
        CK(cudaMemsetAsync(h->iscratch + 2, 0, sizeof(int), sm));
        tile_nnz_max_kernel<<<(unsigned)((tiles + 255) / 256), 256, 0, sm>>>(n, rowptr, tr, tiles, h->iscratch + 2);
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(hs + 2, h->iscratch + 2, sizeof(int), cudaMemcpyDeviceToHost, sm));
        CK(cudaStreamSynchronize(sm));
        if (hs[2] + 3 <= capt) {
            h->cta = true;
            h->cta_tiles = (int)tiles;
        }
    }
    if (h->spmv_variant == 3 && !h->cta) {
        free_problem(h);
        return fail(h, SSTEP_CG_ERR_ARG, "setup: CTA-pipelined SpMV forced but it needs one or two lanes per row, 16 B aligned arrays and "
                                         "tiles (256 rows / 128 or 96 rows) of at most 1797 / 3469 or 2605 entries");
    }
    h->lanes = L;
    return 0;
}

// grids of the Gram / update / init / Alg. 1 kernels
int setup_block_kernels(sstep_cg* h) {
    const int64_t n = h->n;
    const int s = h->s;
    cudaStream_t sm = h->stream;
    h->staged = (h->block_variant == 2) || (h->block_variant == 0 && s >= 5);
    // Gram: staged for every s >= 5; for s = 2..4 on systems of >= 3 M rows, where its few large copies in flight read at 0.955
    // of the read bandwidth against 0.924 for the register kernel (below that the one-CTA-per-SM ramp costs more than it gains;
    // s = 1 gains nothing)
    h->staged_gram = (h->block_variant == 2) || (h->block_variant == 0 && (s >= 5 || (s >= 2 && n >= 3000000)));
    CK(config_spmv(h));
    CK(launch_gram(h, sm, true, nullptr, nullptr, nullptr, nullptr, nullptr, 0));
    CK(launch_update(h, sm, true, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr));
    {
        int64_t want = (n + 255) / 256, cap = (int64_t)h->num_sms * 8;
        h->init_grid = (int)(want < cap ? want : cap);
        want = (n / 2 + 255) / 256;
        if (want < 1) want = 1;
        cap = (int64_t)h->num_sms * 4;  // Alg. 1 kernels: two rows per thread, 4 CTAs per SM
        h->pcg_grid = (int)(want < cap ? want : cap);
    }
    return 0;
}

// eligibility and shape of the resident (whole loop in one cooperative launch) path
int setup_resident(sstep_cg* h) {
    const int64_t n = h->n;
    const int s = h->s;
    cudaStream_t sm = h->stream;
    const int* rowptr = h->rp;
    int hs[4] = {0, 0, 0, 0};
    h->resident = false;
    h->res_grid = 0;
    // (auto: s <= 4 only -- above, the redundant per-CTA reduction of the 2s^2+s partials outweighs the saved launches)
    if (h->resident_opt != 1 && (h->resident_opt == 2 || s <= 4) && h->form == 0 && h->replace_every == 0 && h->method == 0 && n + 4096 < (int64_t(1) << 31)) {
        int coop = 0;
        CK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, h->device));
        int64_t g = (n + 31) / 32;
        if (g > h->num_sms) g = h->num_sms;
        int64_t rpb = ((n + g - 1) / g + 31) / 32 * 32;
        g = (n + rpb - 1) / rpb;
        // (the vectors alone must fit: skips the tile scan for every problem that is far too large)
        if (resident_smem_bytes(s, (int)(rpb < (1 << 20) ? rpb : (1 << 20)), 0) > (size_t)200 * 1024) coop = 0;
        if (coop) {
            CK(cudaMemsetAsync(h->iscratch + 3, 0, sizeof(int), sm));
            tile_nnz_max_kernel<<<(unsigned)((g + 255) / 256), 256, 0, sm>>>(n, rowptr, (int)rpb, g, h->iscratch + 3);
            CK(cudaGetLastError());
            CK(cudaMemcpyAsync(hs + 3, h->iscratch + 3, sizeof(int), cudaMemcpyDeviceToHost, sm));
            CK(cudaStreamSynchronize(sm));
        }
        const int nzcap = (hs[3] + 3) & ~3;
        const size_t bytes = coop ? resident_smem_bytes(s, (int)rpb, nzcap) : 0;
        if (coop && bytes <= (size_t)200 * 1024) {
            h->res_grid = (int)g; h->res_rpb = (int)rpb; h->res_nzcap = nzcap; h->res_smem = bytes;
            h->res_threads = (int)(rpb < 512 ? rpb : 512);
            int occ = 0;
            CK(resident_op(h, sm, 0, 0, &occ));
            h->resident = occ >= 1 && (int64_t)occ * h->num_sms >= g;
        }
        if (!h->resident) h->res_grid = 0;
    }
    if (h->resident_opt == 2 && !h->resident) {
        free_problem(h);
        return fail(h, SSTEP_CG_ERR_ARG, "setup: resident path forced but the problem does not fit shared memory (or form = 1 / replace_every > 0)");
    }
    return 0;
}

// workspaces: R, AR, P, AP, x, r, partial-sum scratch
int setup_workspaces(sstep_cg* h) {
    const int64_t n = h->n;
    const int s = h->s;
    cudaStream_t sm = h->stream;
    const size_t blk = sizeof(double) * (size_t)n * s;
    CK(cudaMalloc(&h->R, blk));
    CK(cudaMalloc(&h->AR, blk));
    CK(cudaMalloc(&h->P, blk));
    CK(cudaMalloc(&h->AP, blk));
    CK(cudaMalloc(&h->x, sizeof(double) * n));
    CK(cudaMalloc(&h->r, sizeof(double) * n));
    size_t np = (size_t)h->gram_grid * (2 * s * s + s);
    if (np < 2 * (size_t)h->update_grid) np = 2 * (size_t)h->update_grid;
    if (np < 2 * (size_t)h->init_grid) np = 2 * (size_t)h->init_grid;
    if (np < 2 * (size_t)h->pcg_grid) np = 2 * (size_t)h->pcg_grid;
    if (np < (size_t)h->res_grid * (2 * s * s + s + 1)) np = (size_t)h->res_grid * (2 * s * s + s + 1);
    CK(cudaMalloc(&h->partials, sizeof(double) * np));
    if (h->resident && h->resident_sync == 0) {  // tagged exchange buffers (resident.cuh, ll_*): all tags start at 0 = "nothing yet"
        h->llR_bytes = sizeof(ulonglong2) * (size_t)n * s;
        h->llPart_bytes = sizeof(ulonglong2) * 2 * (size_t)(2 * s * s + s + 1) * h->res_grid;
        CK(cudaMalloc(&h->llR, h->llR_bytes));
        CK(cudaMalloc(&h->llPart, h->llPart_bytes));
        CK(cudaMalloc(&h->llTot, h->llPart_bytes));
        CK(cudaMemsetAsync(h->llR, 0, h->llR_bytes, sm));
        CK(cudaMemsetAsync(h->llPart, 0, h->llPart_bytes, sm));
        CK(cudaMemsetAsync(h->llTot, 0, h->llPart_bytes, sm));
        h->ll_tag = 0;
    }
    CK(cudaMalloc(&h->mom, sizeof(double) * 2 * s * (size_t)h->spmv_grid));
    CK(cudaMemsetAsync(h->mom, 0, sizeof(double) * 2 * s * (size_t)h->spmv_grid, sm));
    CK(cudaMemsetAsync(h->R, 0, blk, sm));
    CK(cudaMemsetAsync(h->AR, 0, blk, sm));
    CK(cudaMemsetAsync(h->P, 0, blk, sm));
    CK(cudaMemsetAsync(h->AP, 0, blk, sm));
    CK(cudaMemsetAsync(h->st, 0, sizeof(ScgState), sm));
    CK(cudaMemsetAsync(h->st_test, 0, sizeof(ScgState), sm));
    CK(cudaStreamSynchronize(sm));
    return 0;
}

// capture of one outer iteration into a CUDA graph
int setup_graph(sstep_cg* h) {
    if (h->use_graph) {
        const int64_t saved = h->launches;
        for (int attempt = 0; attempt < 2; attempt++) {
            CK(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeRelaxed));
            cudaError_t e = launch_outer(h, h->cap_stream);
            cudaError_t e2 = cudaStreamEndCapture(h->cap_stream, &h->graph);
            h->launches = saved;
            if (e == cudaSuccess && e2 == cudaSuccess) e2 = cudaGraphInstantiate(&h->gexec, h->graph, 0);
            if (e == cudaSuccess && e2 == cudaSuccess) break;
            // a driver that cannot capture / instantiate programmatic edges: once more with plain serialisation
            if (h->graph) cudaGraphDestroy(h->graph);
            h->graph = nullptr;
            h->gexec = nullptr;
            cudaGetLastError();
            if (attempt == 0 && h->pdl) { h->pdl = 0; continue; }
            if (e != cudaSuccess) return fail(h, SSTEP_CG_ERR_CUDA, std::string("graph capture: ") + cudaGetErrorString(e));
            CK(e2);
        }
    }
    return 0;
}

}  // namespace

// =============================================================================================== allocation-free Gram entry
// sstep_cg_gram_noalloc (include/sstep_cg.h): the fused block inner products a2 for callers that cannot call cudaMalloc
// (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  The production gram_kernel<S> needs
// scratch memory -- an ScgState (ticket of the cross-block finish, the finished M, C, m) and the per-block partials
// [2s^2+s][grid] -- which sstep_cg_setup takes from cudaMalloc.  Here the same kernel runs on a file-scope device array
// of a fixed, modest size: NOALLOC_SMAX = 8 (2s^2+s <= 136 entries) x NOALLOC_MAX_BLOCKS = 320 blocks x 8 B = 348 160 B
// + 16 KB for the state = 364 544 B, held by every GPU that loads the library until the process exits.
// In host code the array's NAME is a host-side stand-in, not a device address (a kernel given it faults, or silently
// uses host memory where the GPU can reach it): the address comes from cudaGetSymbolAddress, once per device, with that
// device current, at set-up (sstep_cg_create), and is what the kernels receive.  Every call shares the array, which keeps
// the previous call's contents: the reset kernel clears what must start clean (status, ticket); calls that overlap on the
// GPU (two streams, two handles on one device) race on it.
namespace {

constexpr int NOALLOC_SMAX = 8;
constexpr int NOALLOC_MAX_BLOCKS = 320;
constexpr size_t NOALLOC_STATE_BYTES = 16384;
constexpr size_t NOALLOC_SCRATCH_BYTES =
    NOALLOC_STATE_BYTES + sizeof(double) * (size_t)NOALLOC_MAX_BLOCKS * (2 * NOALLOC_SMAX * NOALLOC_SMAX + NOALLOC_SMAX);
static_assert(sizeof(ScgState) <= NOALLOC_STATE_BYTES, "the state must fit its share of the static scratch");

static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_SCRATCH_BYTES];

constexpr int NOALLOC_MAX_DEVICES = 64;
unsigned char* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};  // device address of g_noalloc_scratch per device (set at create)

// set-up, once per device, with that device current: the DEVICE address of the static array
cudaError_t noalloc_setup_device(int device) {
    if (device < 0 || device >= NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
    if (g_noalloc_ptr[device]) return cudaSuccess;
    void* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    g_noalloc_ptr[device] = static_cast<unsigned char*>(ptr);
    return cudaSuccess;
}

// clears what a call needs clean, whatever the previous call (or an aborted one) left behind
__global__ void noalloc_reset_kernel(ScgState* st) {
    st->status = SCG_RUNNING;  // gram_kernel leaves at once on any other status
    st->ticket_gram = 0;
}

// results out of the static state into the caller's buffers (device code may name the array directly)
__global__ void noalloc_output_kernel(int s, double* __restrict__ M, double* __restrict__ C, double* __restrict__ m) {
    const ScgState* st = reinterpret_cast<const ScgState*>(g_noalloc_scratch);
    for (int e = threadIdx.x; e < s * s; e += blockDim.x) { M[e] = st->M[e]; C[e] = st->C[e]; }
    if ((int)threadIdx.x < s) m[threadIdx.x] = st->m[threadIdx.x];
}

template <int S>
cudaError_t noalloc_gram_S(int num_sms, cudaStream_t sm, int64_t n, const double* R, const double* AR, const double* AP,
                           const double* r, unsigned char* scratch) {
    using Cfg = GramCfg<S>;
    int occ = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, gram_kernel<S>, Cfg::NW * 32, 0);
    if (e != cudaSuccess) return e;
    if (occ < 1) occ = 1;
    int64_t grid = (n + Cfg::RG * 32 - 1) / (Cfg::RG * 32);
    if (grid > (int64_t)occ * num_sms) grid = (int64_t)occ * num_sms;
    if (grid > NOALLOC_MAX_BLOCKS) grid = NOALLOC_MAX_BLOCKS;  // partials [2s^2+s][grid] must fit the static array
    ScgState* st = reinterpret_cast<ScgState*>(scratch);
    double* partials = reinterpret_cast<double*>(scratch + NOALLOC_STATE_BYTES);
    noalloc_reset_kernel<<<1, 1, 0, sm>>>(st);
    gram_kernel<S><<<(unsigned)grid, Cfg::NW * 32, 0, sm>>>(n, R, AR, AP, r, partials, st, /*do_solve=*/0);
    return cudaGetLastError();
}

}  // namespace

// =============================================================================================== C ABI
extern "C" {

int sstep_cg_create(sstep_cg_t** handle, int device, void* cuda_stream) {
    if (!handle) return SSTEP_CG_ERR_ARG;
    *handle = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return SSTEP_CG_ERR_CUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return SSTEP_CG_ERR_CUDA;
    if (prop.major < 10) return SSTEP_CG_ERR_CUDA;  // sm_100a code only: fail loudly elsewhere
    if (cudaSetDevice(device) != cudaSuccess) return SSTEP_CG_ERR_CUDA;
    sstep_cg* h = new sstep_cg();
    h->device = device;
    h->stream = (cudaStream_t)cuda_stream;
    h->num_sms = prop.multiProcessorCount;
    bool ok = cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && noalloc_setup_device(device) == cudaSuccess;  // device address of the static scratch of sstep_cg_gram_noalloc
    ok = ok && cudaMalloc(&h->st, sizeof(ScgState)) == cudaSuccess;
    ok = ok && cudaMalloc(&h->st_test, sizeof(ScgState)) == cudaSuccess;
    ok = ok && cudaMalloc(&h->iscratch, 4 * sizeof(int)) == cudaSuccess;
    ok = ok && cudaMallocHost(&h->h_hdr, 2 * sizeof(Header)) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&h->ev[0], cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&h->ev[1], cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaMemset(h->st, 0, sizeof(ScgState)) == cudaSuccess;
    ok = ok && cudaMemset(h->st_test, 0, sizeof(ScgState)) == cudaSuccess;
    if (!ok) {
        sstep_cg_destroy(h);
        return SSTEP_CG_ERR_CUDA;
    }
    *handle = h;
    return 0;
}

int sstep_cg_destroy(sstep_cg_t* h) {
    if (!h) return SSTEP_CG_ERR_ARG;
    cudaSetDevice(h->device);
    cudaStreamSynchronize(h->stream);
    free_problem(h);
    free_owned(h);
    if (h->st) cudaFree(h->st);
    if (h->st_test) cudaFree(h->st_test);
    if (h->iscratch) cudaFree(h->iscratch);
    if (h->h_hdr) cudaFreeHost(h->h_hdr);
    for (auto& e : h->ev)
        if (e) cudaEventDestroy(e);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    delete h;
    return 0;
}

const char* sstep_cg_last_error(sstep_cg_t* h) { return h ? h->err.c_str() : "null handle"; }

int sstep_cg_set_option(sstep_cg_t* h, const char* key, int64_t value) {
    if (!h || !key) return SSTEP_CG_ERR_ARG;
    const std::string k(key);
    if (k == "basis" && (value == 0 || value == 1)) h->basis = (int)value;
    else if (k == "spmv_variant" && value >= 0 && value <= 3) h->spmv_variant = (int)value;
    else if (k == "spmv_cta_depth" && value >= 2 && value <= 4) h->cta_depth = (int)value;
    else if (k == "spmv_cta_per_sm" && value >= 2 && value <= 3) h->cta_minb = (int)value;
    else if (k == "lanes" && (value == 0 || value == 1 || value == 2 || value == 4 || value == 8 || value == 16 || value == 32))
        h->lanes_opt = (int)value;
    else if (k == "use_graph" && (value == 0 || value == 1)) h->use_graph = (int)value;
    else if (k == "spmv_depth" && value >= 2 && value <= 4) h->spmv_depth = (int)value;
    else if (k == "block_variant" && value >= 0 && value <= 2) h->block_variant = (int)value;
    else if (k == "form" && (value == 0 || value == 1)) h->form = (int)value;
    else if (k == "resident" && value >= 0 && value <= 2) h->resident_opt = (int)value;
    else if (k == "resident_sync" && (value == 0 || value == 1)) h->resident_sync = (int)value;
    else if (k == "reorder" && value >= 0 && value <= 2) h->reorder_opt = (int)value;
    else if (k == "replace_every" && value >= 0 && value <= 1000000) h->replace_every = (int)value;
    else if (k == "method" && (value == 0 || value == 1)) h->method = (int)value;
    else if (k == "pdl" && (value == 0 || value == 1)) h->pdl = (int)value;
    else return fail(h, SSTEP_CG_ERR_ARG, "unknown option or bad value: " + k);
    return 0;
}

int sstep_cg_get_info(sstep_cg_t* h, const char* key, int64_t* value) {
    if (!h || !key || !value) return SSTEP_CG_ERR_ARG;
    const std::string k(key);
    if (k == "lanes") *value = h->lanes;
    else if (k == "spmv_bulk") *value = (h->bulk || h->cta) ? 1 : 0;
    else if (k == "spmv_cta") *value = h->cta ? 1 : 0;
    else if (k == "spmv_grid") *value = h->spmv_grid;
    else if (k == "spmv_depth") *value = h->spmv_depth;
    else if (k == "bulk_cap") *value = h->bulk ? h->bulk_cap : 0;
    else if (k == "block_staged") *value = h->staged ? 1 : 0;
    else if (k == "gram_staged") *value = h->staged_gram ? 1 : 0;
    else if (k == "form") *value = h->form;
    else if (k == "gram_grid") *value = h->gram_grid;
    else if (k == "update_grid") *value = h->update_grid;
    else if (k == "gram_grid_reg") *value = h->gram_grid_reg;
    else if (k == "update_grid_reg") *value = h->update_grid_reg;
    else if (k == "gram_tile_rows") *value = h->gram_tile;
    else if (k == "gram_ring_depth") *value = h->gram_depth;
    else if (k == "update_tile_rows") *value = h->update_tile;
    else if (k == "update_ring_depth") *value = h->update_depth;
    else if (k == "max_row_len") *value = h->max_row_len;
    else if (k == "num_sms") *value = h->num_sms;
    else if (k == "kernels_per_outer") *value = kernels_per_outer(h);
    else if (k == "basis") *value = h->basis;
    else if (k == "launches") *value = h->launches;
    else if (k == "replace_every") *value = h->replace_every;
    else if (k == "method") *value = h->method;
    else if (k == "pdl") *value = h->pdl;
    else if (k == "uniform_diagonal") *value = h->dinv_uniform > 0.0 ? 1 : 0;
    else if (k == "reordered") *value = h->reordered ? 1 : 0;
    else if (k == "cm_levels") *value = h->cm_levels;
    else if (k == "cm_components") *value = h->cm_comps;
    else if (k == "far_permille") *value = h->far_permille;
    else if (k == "resident") *value = h->resident ? 1 : 0;
    else if (k == "resident_grid") *value = h->res_grid;
    else if (k == "resident_sync") *value = h->resident_sync;
    else if (k == "resident_rows_per_block") *value = h->res_rpb;
    else if (k == "resident_smem_bytes") *value = (int64_t)h->res_smem;
    else return fail(h, SSTEP_CG_ERR_ARG, "unknown info key: " + k);
    return 0;
}

int sstep_cg_setup(sstep_cg_t* h, int64_t n, int64_t nnz, const int32_t* rowptr, const int32_t* colidx, const double* vals,
                   int s) {
    if (!h) return SSTEP_CG_ERR_ARG;
    if (n <= 0 || nnz <= 0 || nnz >= (int64_t(1) << 31) || n >= (int64_t(1) << 31) || !rowptr || !colidx || !vals || s < 1 ||
        s > SSTEP_CG_SMAX)
        return fail(h, SSTEP_CG_ERR_ARG, "setup: need n > 0, 0 < nnz < 2^31, non-null CSR arrays, 1 <= s <= 16");
    if (h->form == 1 && h->basis != SSTEP_CG_BASIS_MONOMIAL)
        return fail(h, SSTEP_CG_ERR_ARG, "setup: the moment form (Alg. 5 + Alg. 6) assumes the monomial basis");
    if (h->method == 1 && (s != 1 || h->form != 0 || h->basis != 0 || h->replace_every > 0))
        return fail(h, SSTEP_CG_ERR_ARG, "setup: method = 1 (Alg. 1 PCG) takes s = 1 and none of form / basis / replace_every");
    if (h->form == 1 && h->replace_every > 0)
        return fail(h, SSTEP_CG_ERR_ARG, "setup: residual replacement needs the Gram form (Alg. 6 assumes r = r_prev - AP alpha)");
    CK(cudaSetDevice(h->device));
    CK(cudaStreamSynchronize(h->stream));
    free_problem(h);
    h->n = n; h->nnz = nnz; h->s = s;
    h->rp = rowptr; h->ci = colidx; h->va = vals;

    if (int rc = setup_analyze(h)) return rc;
    if (int rc = setup_reorder(h)) return rc;
    if (int rc = setup_uniform_diagonal(h)) return rc;
    if (int rc = setup_spmv_variant(h)) return rc;
    if (int rc = setup_block_kernels(h)) return rc;
    if (int rc = setup_resident(h)) return rc;
    if (int rc = setup_workspaces(h)) return rc;
    if (int rc = setup_graph(h)) return rc;
    h->ready = true;
    return 0;
}

int sstep_cg_solve_begin(sstep_cg_t* h, const double* b, const double* x0, double rtol) {
    if (!h || !b) return SSTEP_CG_ERR_ARG;
    if (!h->ready) return fail(h, SSTEP_CG_ERR_STATE, "solve: call setup first");
    if (!(rtol >= 0.0)) return fail(h, SSTEP_CG_ERR_ARG, "solve: rtol must be >= 0");
    CK(cudaSetDevice(h->device));
    cudaStream_t sm = h->stream;
    h->t_begin = std::chrono::steady_clock::now();
    h->launches = 0;
    h->graph_launches = 0;
    h->rtol = rtol;
    const size_t blk = sizeof(double) * (size_t)h->n * h->s;
    CK(cudaMemsetAsync(h->P, 0, blk, sm));
    CK(cudaMemsetAsync(h->AP, 0, blk, sm));
    if (h->reordered) {  // b' = Pi b, x0' = Pi x0
        const unsigned g = (unsigned)((h->n + 255) / 256);
        scg_reorder::gather_vec_kernel<<<g, 256, 0, sm>>>(h->n, h->perm, b, h->bperm);
        b = h->bperm;
        if (x0) {
            scg_reorder::gather_vec_kernel<<<g, 256, 0, sm>>>(h->n, h->perm, x0, h->x0perm);
            x0 = h->x0perm;
        }
        CK(cudaGetLastError());
    }
    h->b_cur = b;
    if (x0) {  // r <- A x0 with the production SpMV, then r <- b - r in init_kernel
        CK(launch_spmv(h, sm, x0, h->r, nullptr, nullptr, 0, nullptr));
    }
    init_kernel<<<h->init_grid, 256, 0, sm>>>(h->n, b, x0, x0 ? 1 : 0, h->x, h->r, h->R, h->dinv, h->partials, h->st, h->s, rtol);
    h->launches++;
    CK(cudaGetLastError());
    if (h->method == 1) CK(cudaMemcpyAsync(h->P, h->R, sizeof(double) * h->n, cudaMemcpyDeviceToDevice, sm));  // p_0 = u_0 (Alg. 1 l.3)
    h->in_solve = true;
    return 0;
}

int sstep_cg_iterate(sstep_cg_t* h, int k_outer) {
    if (!h || k_outer < 0) return SSTEP_CG_ERR_ARG;
    if (!h->in_solve) return fail(h, SSTEP_CG_ERR_STATE, "iterate: call solve_begin first");
    if (h->resident) {  // one cooperative launch runs up to k_outer outer iterations (stops on the device at convergence)
        // the grid barrier counts arrivals in 32 bits (resident.cuh): at most 2^31 arrivals per launch, i.e. kcap outer
        // iterations of s + 1 barriers each; longer runs are split into several launches (each re-reads the state and
        // exits at once when the solver has stopped)
        const int64_t kcap = (int64_t(1) << 31) / ((int64_t)h->res_grid * (h->s + 1)) - 1;
        for (int64_t done = 0; done < k_outer;) {
            const int k = (int)((k_outer - done < kcap) ? k_outer - done : kcap);
            if (h->resident_sync == 0) {
                // tags of this launch: ll_tag + 1 .. ll_tag + k + 1; never reused -- before they could wrap, start over from zeroed buffers
                if ((uint64_t)h->ll_tag + (uint64_t)k + 2 >= (uint64_t(1) << 31)) {
                    CK(cudaMemsetAsync(h->llR, 0, h->llR_bytes, h->stream));
                    CK(cudaMemsetAsync(h->llPart, 0, h->llPart_bytes, h->stream));
                    CK(cudaMemsetAsync(h->llTot, 0, h->llPart_bytes, h->stream));
                    h->ll_tag = 0;
                }
            } else {
                CK(cudaMemsetAsync(&h->st->grid_bar, 0, 33 * sizeof(unsigned int), h->stream));
            }
            CK(resident_op(h, h->stream, 1, k, nullptr));
            if (h->resident_sync == 0) h->ll_tag += (unsigned int)k + 2u;
            h->launches++;
            h->graph_launches++;
            done += k;
        }
        return 0;
    }
    for (int i = 0; i < k_outer; i++) {
        if (h->use_graph) {
            CK(cudaGraphLaunch(h->gexec, h->stream));
            h->launches += kernels_per_outer(h);
        } else {
            CK(launch_outer(h, h->stream));
        }
        h->graph_launches++;
        if (h->replace_every > 0 && h->graph_launches % h->replace_every == 0) {
            // residual replacement: y = A x into AR(:,1) (scratch until the next MPK), r <- b - y, R_1, rho, stop test;
            // both kernels exit at once if the update has just declared convergence or a breakdown
            CK(launch_spmv(h, h->stream, h->x, h->AR, nullptr, nullptr, 0, h->st));
            replace_kernel<<<h->init_grid, 256, 0, h->stream>>>(h->n, h->b_cur, h->AR, h->r, h->R, h->dinv, h->partials, h->st);
            CK(cudaGetLastError());
            h->launches++;
        }
    }
    return 0;
}

int sstep_cg_profile_outer(sstep_cg_t* h, int reps, double* ms_host) {
    if (!h || reps < 1 || !ms_host) return SSTEP_CG_ERR_ARG;
    if (!h->in_solve) return fail(h, SSTEP_CG_ERR_STATE, "profile_outer: call solve_begin first");
    if (h->resident) return fail(h, SSTEP_CG_ERR_STATE, "profile_outer: the resident path has no per-kernel launches (set option resident = 1)");
    cudaStream_t sm = h->stream;
    if (h->method == 1) {  // Alg. 1: ms_host[0] = SpMV, [1] = update (K2), [2] = direction (K3)
        cudaEvent_t ev[6];
        for (auto& e : ev) CK(cudaEventCreate(&e));
        ms_host[0] = ms_host[1] = ms_host[2] = 0.0;
        int rc1 = 0;
        for (int rep = 0; rep < reps && rc1 == 0; rep++) {
            if (launch_pcg_iteration(h, sm, ev) != cudaSuccess || cudaStreamSynchronize(sm) != cudaSuccess) { rc1 = SSTEP_CG_ERR_CUDA; break; }
            h->graph_launches++;
            for (int k = 0; k < 3; k++) {
                float ms = 0.f;
                cudaEventElapsedTime(&ms, ev[2 * k], ev[2 * k + 1]);
                ms_host[k] += ms;
            }
        }
        for (auto& e : ev) cudaEventDestroy(e);
        return rc1 ? fail(h, rc1, "profile_outer: CUDA error in the PCG iteration") : 0;
    }
    const int per = h->s + 2;
    const int nev = reps * per * 2;
    cudaEvent_t* evs = new cudaEvent_t[nev];
    for (int i = 0; i < nev; i++) evs[i] = nullptr;
    int rc = 0;
    auto body = [&]() -> int {
        for (int i = 0; i < nev; i++) CK(cudaEventCreate(&evs[i]));
        int e = 0;
        const int64_t n = h->n;
        for (int rep = 0; rep < reps; rep++) {
            for (int j = 0; j < h->s; j++) {
                double* yjac = (j + 1 < h->s) ? h->R + (int64_t)(j + 1) * n : nullptr;
                int mode = 0;
                const double* xprev = nullptr;
                if (h->basis == SSTEP_CG_BASIS_CHEBYSHEV) {
                    mode = (j == 0) ? 1 : 2;
                    if (j > 0) xprev = h->R + (int64_t)(j - 1) * n;
                }
                CK(cudaEventRecord(evs[e++], sm));
                double* mom_a = h->form ? h->mom + (int64_t)(2 * j + 1) * h->spmv_grid : nullptr;
                double* mom_b = (h->form && j + 1 < h->s) ? h->mom + (int64_t)(2 * j + 2) * h->spmv_grid : nullptr;
                CK(launch_spmv(h, sm, h->R + (int64_t)j * n, h->AR + (int64_t)j * n, yjac, xprev, mode, h->st, mom_a, mom_b));
                CK(cudaEventRecord(evs[e++], sm));
            }
            CK(cudaEventRecord(evs[e++], sm));
            CK(h->form ? launch_sw(h, sm, h->st, 1) : launch_gram(h, sm, false, h->R, h->AR, h->AP, h->r, h->st, 1));
            CK(cudaEventRecord(evs[e++], sm));
            CK(cudaEventRecord(evs[e++], sm));
            CK(launch_update(h, sm, false, h->R, h->AR, h->P, h->AP, h->x, h->r, h->st->beta, h->st->alpha, h->st, nullptr));
            CK(cudaEventRecord(evs[e++], sm));
            h->graph_launches++;
        }
        CK(cudaStreamSynchronize(sm));
        ms_host[0] = ms_host[1] = ms_host[2] = 0.0;
        e = 0;
        for (int rep = 0; rep < reps; rep++)
            for (int k = 0; k < per; k++) {
                float ms = 0.f;
                CK(cudaEventElapsedTime(&ms, evs[e], evs[e + 1]));
                e += 2;
                ms_host[k < h->s ? 0 : (k == h->s ? 1 : 2)] += ms;
            }
        return 0;
    };
    rc = body();
    for (int i = 0; i < nev; i++)
        if (evs[i]) cudaEventDestroy(evs[i]);
    delete[] evs;
    return rc;
}

int sstep_cg_solve_peek(sstep_cg_t* h, sstep_cg_result* out) {
    if (!h || !out) return SSTEP_CG_ERR_ARG;
    if (!h->in_solve) return fail(h, SSTEP_CG_ERR_STATE, "solve_peek: call solve_begin first");
    cudaStream_t sm = h->stream;
    CK(cudaMemcpyAsync(&h->h_hdr[0], h->st, sizeof(Header), cudaMemcpyDeviceToHost, sm));
    CK(cudaStreamSynchronize(sm));
    const Header hd = h->h_hdr[0];
    out->status = hd.status;  // SSTEP_CG_RUNNING while the stop test has not fired
    out->outer_iters = hd.k;
    out->cg_equiv_iters = (int64_t)hd.k * h->s;
    out->r0_norm = sqrt(hd.rho0);
    out->relres = hd.rho0 > 0.0 ? sqrt(hd.rho) / sqrt(hd.rho0) : 0.0;
    out->solve_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - h->t_begin).count();
    out->kernel_launches = h->launches;
    return 0;
}

int sstep_cg_solve_end(sstep_cg_t* h, double* x, sstep_cg_result* out) {
    if (!h) return SSTEP_CG_ERR_ARG;
    if (!h->in_solve) return fail(h, SSTEP_CG_ERR_STATE, "solve_end: call solve_begin first");
    cudaStream_t sm = h->stream;
    if (x && h->reordered) {  // x = Pi^T x'
        scg_reorder::scatter_vec_kernel<<<(unsigned)((h->n + 255) / 256), 256, 0, sm>>>(h->n, h->perm, h->x, x);
        CK(cudaGetLastError());
    } else if (x) {
        CK(cudaMemcpyAsync(x, h->x, sizeof(double) * h->n, cudaMemcpyDeviceToDevice, sm));
    }
    CK(cudaMemcpyAsync(&h->h_hdr[0], h->st, sizeof(Header), cudaMemcpyDeviceToHost, sm));
    CK(cudaStreamSynchronize(sm));
    h->in_solve = false;
    const Header hd = h->h_hdr[0];
    const int status = (hd.status == SCG_RUNNING) ? SSTEP_CG_MAXIT : hd.status;
    if (out) {
        out->status = status;
        out->outer_iters = hd.k;
        out->cg_equiv_iters = (int64_t)hd.k * h->s;
        out->r0_norm = sqrt(hd.rho0);
        out->relres = hd.rho0 > 0.0 ? sqrt(hd.rho) / sqrt(hd.rho0) : 0.0;
        out->solve_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - h->t_begin).count();
        out->kernel_launches = h->launches;
    }
    return status;
}

int sstep_cg_solve(sstep_cg_t* h, const double* b, const double* x0, double* x, double rtol, int maxit, sstep_cg_result* out) {
    if (!h || !x || maxit < 0) return SSTEP_CG_ERR_ARG;
    int rc = sstep_cg_solve_begin(h, b, x0, rtol);
    if (rc) return rc;
    cudaStream_t sm = h->stream;
    if (h->resident) {  // the whole loop is one launch; the stop test runs on the device
        rc = sstep_cg_iterate(h, maxit);
        if (rc) return rc;
        return sstep_cg_solve_end(h, x, out);
    }
    // Replay the outer-iteration graph in chunks; two chunks are kept in flight so the device never waits for the
    // host.  Iterations enqueued after convergence exit on the device flag (a few microseconds each).
    const int chunk = h->n >= (int64_t(1) << 21) ? 2 : 8;
    int launched = 0, slot = 0;
    bool pending[2] = {false, false};
    bool done = false;
    while (true) {
        if (!done && launched < maxit) {
            const int k = (maxit - launched < chunk) ? maxit - launched : chunk;
            rc = sstep_cg_iterate(h, k);
            if (rc) return rc;
            launched += k;
            CK(cudaMemcpyAsync(&h->h_hdr[slot], h->st, sizeof(Header), cudaMemcpyDeviceToHost, sm));
            CK(cudaEventRecord(h->ev[slot], sm));
            pending[slot] = true;
            slot ^= 1;
        }
        if (pending[slot]) {  // the older of the two chunks
            CK(cudaEventSynchronize(h->ev[slot]));
            pending[slot] = false;
            if (h->h_hdr[slot].status != SCG_RUNNING) done = true;
        } else if (done || launched >= maxit) {
            if (pending[slot ^ 1]) {
                CK(cudaEventSynchronize(h->ev[slot ^ 1]));
                pending[slot ^ 1] = false;
            }
            break;
        }
    }
    return sstep_cg_solve_end(h, x, out);
}

int sstep_cg_solve_host(sstep_cg_t* h, int64_t n, int64_t nnz, const int32_t* rp, const int32_t* ci, const double* va,
                        const double* b, const double* x0, double* x, int s, double rtol, int maxit, sstep_cg_result* out) {
    if (!h || !rp || !ci || !va || !b || !x || n <= 0 || nnz <= 0) return SSTEP_CG_ERR_ARG;
    CK(cudaSetDevice(h->device));
    cudaStream_t sm = h->stream;
    CK(cudaStreamSynchronize(sm));
    free_problem(h);
    if (!(h->own_x && h->own_n == n && h->own_nnz == nnz)) {  // a repeated call with the same sizes keeps its device copies' storage
        free_owned(h);
        CK(cudaMalloc(&h->own_rp, sizeof(int) * (n + 1)));
        CK(cudaMalloc(&h->own_ci, sizeof(int) * nnz));
        CK(cudaMalloc(&h->own_va, sizeof(double) * nnz));
        CK(cudaMalloc(&h->own_b, sizeof(double) * n));
        CK(cudaMalloc(&h->own_x, sizeof(double) * n));
        h->own_n = n;
        h->own_nnz = nnz;
    }
    CK(cudaMemcpyAsync(h->own_rp, rp, sizeof(int) * (n + 1), cudaMemcpyHostToDevice, sm));
    CK(cudaMemcpyAsync(h->own_ci, ci, sizeof(int) * nnz, cudaMemcpyHostToDevice, sm));
    CK(cudaMemcpyAsync(h->own_va, va, sizeof(double) * nnz, cudaMemcpyHostToDevice, sm));
    CK(cudaMemcpyAsync(h->own_b, b, sizeof(double) * n, cudaMemcpyHostToDevice, sm));
    if (x0) CK(cudaMemcpyAsync(h->own_x, x0, sizeof(double) * n, cudaMemcpyHostToDevice, sm));
    int rc = sstep_cg_setup(h, n, nnz, h->own_rp, h->own_ci, h->own_va, s);
    if (rc) return rc;
    rc = sstep_cg_solve(h, h->own_b, x0 ? h->own_x : nullptr, h->own_x, rtol, maxit, out);
    if (rc < 0) return rc;
    CK(cudaMemcpyAsync(x, h->own_x, sizeof(double) * n, cudaMemcpyDeviceToHost, sm));
    CK(cudaStreamSynchronize(sm));
    return rc;
}

// ---------------------------------------------------------------- measurement aid (measure.cuh)
int sstep_cg_measure_bandwidth(sstep_cg_t* h, int variant, int64_t bytes, int passes, int reps, double* gbs_out) {
    if (!h || !gbs_out || variant < 0 || variant > 5 || bytes < (1 << 20) || passes < 1 || reps < 1) return SSTEP_CG_ERR_ARG;
    if (h->in_solve) return fail(h, SSTEP_CG_ERR_STATE, "measure_bandwidth: a solve is in progress");
    CK(cudaSetDevice(h->device));
    cudaStream_t sm = h->stream;
    bytes &= ~(int64_t)8191;
    unsigned char *src = nullptr, *dst = nullptr;
    double* sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = 0;
    auto body = [&]() -> int {
        CK(cudaMalloc(&src, (size_t)bytes));
        CK(cudaMalloc(&sink, sizeof(double)));
        CK(cudaMemsetAsync(src, 0, (size_t)bytes, sm));
        if (variant == 2) {
            CK(cudaMalloc(&dst, (size_t)bytes));
            CK(cudaMemsetAsync(dst, 0, (size_t)bytes, sm));
        }
        CK(cudaEventCreate(&e0));
        CK(cudaEventCreate(&e1));
        int occ = 1;
        if (variant == 0) CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, measure_read_ldg_kernel, 256, 0));
        if (variant == 2) CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, measure_copy_kernel, 256, 0));
        const int grid = (occ < 1 ? 1 : occ) * h->num_sms;
        double best = 0.0, sum = 0.0;
        for (int rep = -1; rep < reps; rep++) {  // rep -1 = warm-up
            CK(cudaEventRecord(e0, sm));
            if (variant == 0) measure_read_ldg_kernel<<<grid, 256, 0, sm>>>((const double2*)src, bytes / 16, passes, sink);
            else if (variant == 2) measure_copy_kernel<<<grid, 256, 0, sm>>>((const double2*)src, (double2*)dst, bytes / 16, passes);
            else if (variant == 1) CK((launch_measure_bulk<2, 4096, 8>(h->num_sms, 3, sm, src, bytes, passes, sink)));   // 48 copies in flight per SM
            else if (variant == 3) CK((launch_measure_bulk<4, 2048, 8>(h->num_sms, 3, sm, src, bytes, passes, sink)));   // 96
            else if (variant == 4) CK((launch_measure_bulk<2, 8192, 4>(h->num_sms, 3, sm, src, bytes, passes, sink)));   // 24
            else CK((launch_measure_bulk<2, 4096, 8>(h->num_sms, 2, sm, src, bytes, passes, sink)));                     // 32
            CK(cudaGetLastError());
            CK(cudaEventRecord(e1, sm));
            CK(cudaEventSynchronize(e1));
            float ms = 0.f;
            CK(cudaEventElapsedTime(&ms, e0, e1));
            if (rep < 0) continue;
            const double gbs = (variant == 2 ? 2.0 : 1.0) * (double)bytes * passes / (ms * 1e-3) / 1e9;
            sum += gbs;
            if (gbs > best) best = gbs;
        }
        gbs_out[0] = best;
        gbs_out[1] = sum / reps;
        return 0;
    };
    rc = body();
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (src) cudaFree(src);
    if (dst) cudaFree(dst);
    if (sink) cudaFree(sink);
    return rc;
}

// ---------------------------------------------------------------- test hooks (production kernels, caller's buffers)
static int hook_prepare(sstep_cg* h) {
    if (!h->ready) return fail(h, SSTEP_CG_ERR_STATE, "test hook: call setup first");
    if (h->in_solve) return fail(h, SSTEP_CG_ERR_STATE, "test hook: a solve is in progress");
    CK(cudaSetDevice(h->device));
    // st_test: status = running, tickets 0, rho0 = 0 (stop test never fires), rtol = 0
    ScgState init;
    memset(&init, 0, sizeof init);
    init.status = SCG_RUNNING;
    CK(cudaMemcpyAsync(h->st_test, &init, sizeof(Header) /* header only; tickets stay 0 */, cudaMemcpyHostToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return 0;
}

int sstep_cg_get_permutation(sstep_cg_t* h, int32_t* perm_out) {
    if (!h || !perm_out) return SSTEP_CG_ERR_ARG;
    if (!h->ready) return fail(h, SSTEP_CG_ERR_STATE, "get_permutation: call setup first");
    CK(cudaSetDevice(h->device));
    if (h->reordered) {
        CK(cudaMemcpyAsync(perm_out, h->perm, sizeof(int) * (size_t)h->n, cudaMemcpyDeviceToDevice, h->stream));
    } else {
        iota_kernel<<<(unsigned)((h->n + 255) / 256), 256, 0, h->stream>>>(h->n, perm_out);
        CK(cudaGetLastError());
    }
    CK(cudaStreamSynchronize(h->stream));
    return 0;
}

int sstep_cg_test_read_state(sstep_cg_t* h, const char* name, double* out, int64_t count) {
    if (!h || !name || !out) return SSTEP_CG_ERR_ARG;
    if (!h->ready) return fail(h, SSTEP_CG_ERR_STATE, "test_read_state: call setup first");
    CK(cudaSetDevice(h->device));
    const std::string k(name);
    const int64_t ns = h->n * h->s, ss = (int64_t)h->s * h->s;
    const double* src = nullptr;
    int64_t want = 0;
    if (k == "R") { src = h->R; want = ns; }
    else if (k == "AR") { src = h->AR; want = ns; }
    else if (k == "P") { src = h->P; want = ns; }
    else if (k == "AP") { src = h->AP; want = ns; }
    else if (k == "x") { src = h->x; want = h->n; }
    else if (k == "r") { src = h->r; want = h->n; }
    else if (k == "M") { src = h->st->M; want = ss; }
    else if (k == "C") { src = h->st->C; want = ss; }
    else if (k == "W") { src = h->st->W; want = ss; }
    else if (k == "beta") { src = h->st->beta; want = ss; }
    else if (k == "m") { src = h->st->m; want = h->s; }
    else if (k == "alpha") { src = h->st->alpha; want = h->s; }
    else return fail(h, SSTEP_CG_ERR_ARG, "test_read_state: unknown array " + k);
    if (count != want) return fail(h, SSTEP_CG_ERR_ARG, "test_read_state: wrong element count for " + k);
    CK(cudaMemcpyAsync(out, src, sizeof(double) * want, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return 0;
}

int sstep_cg_test_spmv(sstep_cg_t* h, const double* x, double* y, double* yjac) {
    if (!h || !x || !y) return SSTEP_CG_ERR_ARG;
    int rc = hook_prepare(h);
    if (rc) return rc;
    CK(launch_spmv(h, h->stream, x, y, yjac, nullptr, 0, h->st_test));
    CK(cudaStreamSynchronize(h->stream));
    return 0;
}

int sstep_cg_test_mpk(sstep_cg_t* h, const double* r, double* R, double* AR) {
    if (!h || !r || !R || !AR) return SSTEP_CG_ERR_ARG;
    int rc = hook_prepare(h);
    if (rc) return rc;
    // R(:,1) = D^-1 r through the production init kernel (b = r, x0 = 0); x and r outputs go to the workspaces
    init_kernel<<<h->init_grid, 256, 0, h->stream>>>(h->n, r, nullptr, 0, h->x, h->r, R, h->dinv, h->partials, h->st_test, h->s, 0.0);
    CK(cudaGetLastError());
    CK(launch_mpk(h, h->stream, R, AR, h->st_test));
    CK(cudaStreamSynchronize(h->stream));
    return 0;
}

int sstep_cg_test_mpk_moments(sstep_cg_t* h, const double* r, double* R, double* AR, double* vm) {
    if (!h || !r || !R || !AR || !vm) return SSTEP_CG_ERR_ARG;
    int rc = hook_prepare(h);
    if (rc) return rc;
    if (!h->form) return fail(h, SSTEP_CG_ERR_STATE, "test_mpk_moments: set option form = 1 before setup");
    init_kernel<<<h->init_grid, 256, 0, h->stream>>>(h->n, r, nullptr, 0, h->x, h->r, R, h->dinv, h->partials, h->st_test, h->s, 0.0);
    CK(cudaGetLastError());
    CK(launch_mpk(h, h->stream, R, AR, h->st_test));
    CK(launch_sw(h, h->stream, h->st_test, 0));
    CK(cudaMemcpyAsync(vm, h->st_test->vm, sizeof(double) * 2 * h->s, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return 0;
}

int sstep_cg_test_sw(sstep_cg_t* h, const double* vm, int first, double* beta, double* alpha, double* W, int32_t* status_out) {
    if (!h || !vm || !beta || !alpha || !W || !status_out) return SSTEP_CG_ERR_ARG;
    int rc = hook_prepare(h);
    if (rc) return rc;
    sw_test_kernel<<<1, 32, 0, h->stream>>>(h->s, first, vm, beta, alpha, W, status_out);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(h->stream));
    return 0;
}

int sstep_cg_test_gram(sstep_cg_t* h, const double* R, const double* AR, const double* AP, const double* r, double* M,
                       double* C, double* m) {
    if (!h || !R || !AR || !AP || !r || !M || !C || !m) return SSTEP_CG_ERR_ARG;
    int rc = hook_prepare(h);
    if (rc) return rc;
    const int s = h->s;
    CK(launch_gram(h, h->stream, false, R, AR, AP, r, h->st_test, 0));
    CK(cudaMemcpyAsync(M, h->st_test->M, sizeof(double) * s * s, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaMemcpyAsync(C, h->st_test->C, sizeof(double) * s * s, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaMemcpyAsync(m, h->st_test->m, sizeof(double) * s, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return 0;
}

int sstep_cg_test_small_solve(sstep_cg_t* h, const double* M, const double* C, const double* m, const double* Wprev,
                              double* beta, double* alpha, double* W, int32_t* status_out) {
    if (!h || !M || !C || !m || !Wprev || !beta || !alpha || !W || !status_out) return SSTEP_CG_ERR_ARG;
    int rc = hook_prepare(h);
    if (rc) return rc;
    small_solve_kernel<<<1, 32, 0, h->stream>>>(h->s, M, C, m, Wprev, nullptr, beta, alpha, W, nullptr, status_out);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(h->stream));
    return 0;
}

int sstep_cg_test_small_solve_carried(sstep_cg_t* h, const double* M, const double* C, const double* m, const double* Lprev,
                                      double* beta, double* alpha, double* W, double* Lout, int32_t* status_out) {
    if (!h || !M || !C || !m || !Lprev || !beta || !alpha || !W || !Lout || !status_out) return SSTEP_CG_ERR_ARG;
    int rc = hook_prepare(h);
    if (rc) return rc;
    small_solve_kernel<<<1, 32, 0, h->stream>>>(h->s, M, C, m, nullptr, Lprev, beta, alpha, W, Lout, status_out);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(h->stream));
    return 0;
}

int sstep_cg_test_division(sstep_cg_t* h, int64_t n, const double* a, const double* b, double* q) {
    if (!h || n < 0 || (n > 0 && (!a || !b || !q))) return SSTEP_CG_ERR_ARG;
    if (n == 0) return 0;
    CK(cudaSetDevice(h->device));
    const int blocks = (int)std::min<int64_t>((n + 255) / 256, (int64_t)h->num_sms * 8);
    division_test_kernel<<<blocks, 256, 0, h->stream>>>(n, a, b, q);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(h->stream));
    return 0;
}

int sstep_cg_test_update(sstep_cg_t* h, double* R, const double* AR, double* P, double* AP, double* x, double* r,
                         const double* beta, const double* alpha, double* rho_out) {
    if (!h || !R || !AR || !P || !AP || !x || !r || !beta || !alpha) return SSTEP_CG_ERR_ARG;
    int rc = hook_prepare(h);
    if (rc) return rc;
    CK(launch_update(h, h->stream, false, R, AR, P, AP, x, r, beta, alpha, h->st_test, rho_out));
    CK(cudaStreamSynchronize(h->stream));
    return 0;
}

int sstep_cg_gram_noalloc(sstep_cg_t* h, int64_t n, int s, const double* R, const double* AR, const double* AP,
                          const double* r, double* M, double* C, double* m) {
    if (!h || !R || !AR || !AP || !r || !M || !C || !m) return SSTEP_CG_ERR_ARG;
    if (s < 1 || s > NOALLOC_SMAX)
        return fail(h, SSTEP_CG_ERR_ARG, "gram_noalloc: block size s must be 1..8 (the static scratch holds 2s^2+s <= 136 entries per "
                                         "block; use sstep_cg_setup + the solver, or sstep_cg_test_gram, for larger s)");
    if (n < 1 || n >= (int64_t(1) << 40)) return fail(h, SSTEP_CG_ERR_ARG, "gram_noalloc: need 1 <= n < 2^40 rows");
    unsigned char* scratch = (h->device < NOALLOC_MAX_DEVICES) ? g_noalloc_ptr[h->device] : nullptr;
    if (!scratch) return fail(h, SSTEP_CG_ERR_STATE, "gram_noalloc: the static scratch of this device was not set up (sstep_cg_create does it)");
    cudaStream_t sm = h->stream;
    cudaError_t e = cudaSuccess;
    switch (s) {
        case 1: e = noalloc_gram_S<1>(h->num_sms, sm, n, R, AR, AP, r, scratch); break;
        case 2: e = noalloc_gram_S<2>(h->num_sms, sm, n, R, AR, AP, r, scratch); break;
        case 3: e = noalloc_gram_S<3>(h->num_sms, sm, n, R, AR, AP, r, scratch); break;
        case 4: e = noalloc_gram_S<4>(h->num_sms, sm, n, R, AR, AP, r, scratch); break;
        case 5: e = noalloc_gram_S<5>(h->num_sms, sm, n, R, AR, AP, r, scratch); break;
        case 6: e = noalloc_gram_S<6>(h->num_sms, sm, n, R, AR, AP, r, scratch); break;
        case 7: e = noalloc_gram_S<7>(h->num_sms, sm, n, R, AR, AP, r, scratch); break;
        default: e = noalloc_gram_S<8>(h->num_sms, sm, n, R, AR, AP, r, scratch); break;
    }
    if (e != cudaSuccess) return fail(h, SSTEP_CG_ERR_CUDA, std::string("gram_noalloc: ") + cudaGetErrorString(e));
    noalloc_output_kernel<<<1, 64, 0, sm>>>(s, M, C, m);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h, SSTEP_CG_ERR_CUDA, std::string("gram_noalloc: ") + cudaGetErrorString(e));
    return 0;  // asynchronous on the handle's stream, like every kernel launch
}

}  // extern "C"

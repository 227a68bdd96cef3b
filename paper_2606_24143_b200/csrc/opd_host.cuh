// Host-side plumbing of libopd: handle, workspace planner, TMA descriptor encoding, GEMM launcher.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <string>
#include <utility>

#include "../../include/opd.h"
#include "opd_bwd_kernel.cuh"
#include "opd_estimators.cuh"
#include "opd_sparse_bwd.cuh"
#include "opd_producer.cuh"

struct opd_handle_s {
    int device = 0;
    int num_sms = 0;
    int cg = 2;                    // tcgen05 cta_group of the GEMM core: 2 = CTA pairs (default), 1 = single CTAs (OPD_CTA_GROUP)
    bool arch_ok = false;
    int l2_bytes = 0, l2_persist_max = 0, l2_window_max = 0;   // L2 size, largest persisting carve-out, largest access-policy window
    size_t l2_persist = 0;         // persisting carve-out this handle asked for (cudaLimitPersistingL2CacheSize)
    void* ws = nullptr;            // workspace in use
    size_t ws_bytes = 0;
    bool ws_owned = false;
    std::string err;
    // host-entry staging buffers (opd_loss_fwd_bwd_host)
    void* stage[2] = {nullptr, nullptr};
    size_t stage_bytes[2] = {0, 0};
    cudaStream_t host_stream = nullptr, host_in = nullptr, host_out = nullptr;   // compute, copy-in, copy-out
    cudaEvent_t ev_in[2] = {}, ev_c[2] = {}, ev_out[2] = {};
    size_t slot_h2d[2] = {0, 0}, slot_d2h[2] = {0, 0};
    bool slot_busy[2] = {false, false};
    int bwd_grid[3][2] = {{0, 0}, {0, 0}, {0, 0}};   // [cta group][dense]: grid of the persistent backward on THIS device (0 = not computed)
    // stats of the last call
    int n_kernels = 0, n_gemm = 0, super_rows = 0, super_cols = 0;
    cudaEvent_t* phase_events = nullptr;
    float* diag_rho = nullptr; long diag_ld_rho = 0; float* diag_var1 = nullptr;   // opd_set_diagnostics
    int diag_rows = 0, diag_cols = 0;                                               // capacity of the diagnostics arrays
    int seq_n = 0; const int* seq_cu = nullptr;                                     // opd_set_seq_diagnostics
    float *seq_mean_m = nullptr, *seq_mean_1 = nullptr, *seq_var_m = nullptr;
};

namespace opd {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// bf16 tensor [planes][rows][inner] (inner contiguous), 128-byte swizzled boxes of 64 x box_rows x 1
inline bool make_map(CUtensorMap* m, const void* base, uint64_t inner, uint64_t rows, uint64_t planes,
                     uint64_t row_stride_bytes, uint64_t plane_stride_bytes, uint32_t box_rows) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return false;
    cuuint64_t dims[3] = {inner, rows, planes};
    cuuint64_t strides[2] = {row_stride_bytes, plane_stride_bytes};
    cuuint32_t box[3] = {64, box_rows, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// fp32 matrix [rows][cols] (row stride in bytes), 128-byte swizzled boxes of 32 x 32 (epilogue store / reduce-add)
inline bool make_map_f32(CUtensorMap* m, const void* base, uint64_t cols, uint64_t rows, uint64_t row_stride_bytes) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return false;
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {row_stride_bytes};
    cuuint32_t box[2] = {32, 32};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline int ceil_div(int a, int b) { return (a + b - 1) / b; }

// ---------------------------------------------------------------- workspace plan
struct Plan {
    int T, d, V, C, planes;
    int t_pad;            // T rounded up to 128
    int num_n;            // vocabulary tiles of 256
    int Tb, Vb;           // backward super-tile (rows of tokens x vocabulary columns), multiples of 128 / 256
    int est_blocks;
    size_t off_nlive, off_badidx, off_live_rows, off_xc, off_wsplit, off_sorted, off_perm, off_zc, off_beta,
           off_partials, off_lse2, off_coef, off_gs, off_dxacc, off_block_sums, off_counters, off_wt, off_skeys, off_shist, off_gwseg, off_gw32,
           off_seq_l1, off_seq_var1, total;
    bool sparse_bwd;      // alpha == 0 on every row: gradients live on the cached columns only (no dense backward)
    int n_super;          // number of backward super-tiles (upper bound)
    int gs_bufs;          // ring depth of the G super-tile buffer
    size_t xc_plane, w_plane, gs_plane;   // elements per plane
    size_t sort_n; int sort_blocks;       // sparse backward: entries to sort, blocks of the radix sort
    size_t dv_bytes;      // bytes of the items of size O(d*V) (bf16 planes of an fp32 W, transposed W, fp32 sums behind a bf16 grad_W):
                          // weight-sized, not logits-sized, so they do not count against the T x V budget of make_plan
};

inline int env_int(const char* name, int dflt) {
    const char* s = std::getenv(name);
    return (s && *s) ? std::atoi(s) : dflt;
}

// 0 = normal, 1 = evict first, 2 = evict last
inline unsigned long long hint_policy(int code) {
    return code == 1 ? L2_EVICT_FIRST : (code == 2 ? L2_EVICT_LAST : L2_EVICT_NORMAL);
}

inline int cta_group_setting() {
    const int cg = env_int("OPD_CTA_GROUP", 2);
    return cg == 1 ? 1 : 2;
}

// vb / gbufs: vocabulary columns per super-tile and depth of the G ring (chosen by make_plan)
inline Plan make_plan_cfg(int T, int d, int V, int C, int fp32, unsigned flags, int mode, int vb, int gbufs) {
    Plan p{};
    p.T = T; p.d = d; p.V = V; p.C = C; p.planes = fp32 ? 3 : 1;
    const int TM = BM * cta_group_setting();              // tile rows of the GEMM core (CTA or CTA pair)
    p.t_pad = ceil_div(T, TM) * TM;
    p.num_n = ceil_div(V, BN);
    // Super-tile of the backward: up to 4608 (4736 for single-CTA tiles) token rows x 4096 vocabulary columns = 288 pair
    // tiles (592 CTA tiles) per G re-formation; the bf16 G super-tile (at most 36-37 MiB) is consumed out of L2.  Among
    // the row counts between 3584 and the maximum the one that wastes the fewest padded rows in the last token
    // super-tile is taken (T = 32768 or 65536: 4096 rows, i.e. equal super-tiles; measured 2% faster than 4608 at C4).
    const int tb_max = TM == 256 ? 18 * 256 : 37 * BM;
    int tb = env_int("OPD_TB", 0);
    if (tb <= 0) {
        tb = tb_max;
        long best_waste = -1;
        for (int cand = tb_max; cand >= 3584 && p.t_pad > tb_max; cand -= TM) {
            const long waste = (long)ceil_div(p.t_pad, cand) * cand - p.t_pad;
            if (best_waste < 0 || waste < best_waste) { best_waste = waste; tb = cand; }
        }
    }
    p.Tb = std::min(p.t_pad, std::max(TM, tb / TM * TM));
    p.Vb = std::min(p.num_n * BN, std::max(BN, vb / BN * BN));
    p.est_blocks = ceil_div(T, 128);
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes, 1024); return r; };
    p.off_nlive = take(4);
    p.off_badidx = take(4);
    p.off_live_rows = take(sizeof(int) * (size_t)p.t_pad);
    p.xc_plane = (size_t)p.t_pad * d;
    p.off_xc = take(2 * p.xc_plane * p.planes);
    p.w_plane = (size_t)d * V;
    p.off_wsplit = take(fp32 ? 2 * p.w_plane * 3 : 0);
    p.off_sorted = take(sizeof(int) * (size_t)p.t_pad * C);
    p.off_perm = take((size_t)p.t_pad * C);
    p.off_zc = take(sizeof(float) * (size_t)p.t_pad * C);
    p.off_beta = take(sizeof(float) * (size_t)p.t_pad * C);
    p.off_lse2 = take(sizeof(float) * (size_t)p.t_pad);
    p.off_coef = take(sizeof(float) * (size_t)p.t_pad);
    const bool bwd = !(flags & OPD_F_FWD_ONLY);
    p.sparse_bwd = (mode == OPD_RKL_TOPK || (mode == OPD_FKL_TOPK && (flags & OPD_F_RENORM_STUDENT)));
#ifdef OPD_EXPERIMENTS
    if (env_int("OPD_DENSE_BWD", 0)) p.sparse_bwd = false;     // timing experiment: run the dense backward anyway
#endif
    // sparse backward: with [d,V] storage W is read through a [V,d] transposed copy (contiguous d-vectors per cached
    // column; callers that store W as [V,d] like lm_head.weight need none); sort buffers of the T*C (column, entry) pairs
    p.off_wt = take(bwd && p.sparse_bwd ? (size_t)d * V * (fp32 ? 4 : 2) : 0);
    p.sort_n = (size_t)p.t_pad * C;
    p.sort_blocks = (int)((p.sort_n + RS_TILE - 1) / RS_TILE);
    p.off_skeys = take(bwd && p.sparse_bwd ? 4 * sizeof(uint32_t) * p.sort_n : 0);          // keys / values, ping-pong
    p.off_shist = take(bwd && p.sparse_bwd ? sizeof(uint32_t) * 256 * (size_t)p.sort_blocks : 0);
    p.off_gwseg = take(bwd && p.sparse_bwd ? sizeof(float) * (p.sort_n / GW_SEG) * (size_t)d : 0);   // per-segment partial sums (hot columns)
    p.off_gw32 = take(bwd && (flags & OPD_F_GRADW_BF16) ? (size_t)d * V * 4 : 0);      // fp32 sums behind a bf16 grad_W
    p.off_seq_l1 = take(sizeof(float) * (size_t)p.t_pad);                               // per-token terms of opd_set_seq_diagnostics
    p.dv_bytes = (p.off_sorted - p.off_wsplit) + (p.off_skeys - p.off_wt) + (p.off_seq_l1 - p.off_gw32);   // each followed by the next take()
    p.off_seq_var1 = take(sizeof(float) * (size_t)p.t_pad);
    p.gs_plane = (size_t)p.Tb * p.Vb;
    p.gs_bufs = std::min(3, std::max(2, gbufs));
    p.n_super = ceil_div(p.t_pad, p.Tb) * ceil_div(V, p.Vb);
    p.off_counters = take(bwd ? sizeof(int) * (3 * (size_t)p.n_super + 1) : 0);      // g_done, dx_done, dw_done, tile ticket
    // The per-tile LSE partials are dead once the estimators have run, the G ring and the grad_hidden partial
    // sums only live in the backward: they share one region.
    const size_t partial_bytes = align_up(sizeof(float2) * (size_t)p.num_n * p.t_pad, 1024);
    const size_t gs_bytes = bwd && !p.sparse_bwd ? align_up(2 * p.gs_plane * p.planes * p.gs_bufs, 1024) : 0;
    const size_t dx_bytes = bwd && !p.sparse_bwd ? align_up(sizeof(float) * (size_t)p.Tb * d, 1024) : 0;
    const size_t region = take(std::max(partial_bytes, gs_bytes + dx_bytes));
    p.off_partials = region;
    p.off_gs = region;
    p.off_dxacc = region + gs_bytes;
    p.off_block_sums = take(sizeof(double) * (size_t)p.est_blocks);
    p.total = o;
    return p;
}

// Chooses the super-tile width Vb (= K depth of a grad_hidden tile) and the depth of the G ring under a workspace budget of
// 4.8% of the bf16 logits (no buffer of the order of T x V), from the sweeps of profiles/r02_experiments.md.
// The budget is applied to what grows with T (and with the super-tile): the weight-sized items (Plan::dv_bytes: the bf16
// planes of an fp32 W, the transposed W of the sparse backward, the fp32 sums behind a bf16 grad_W) are the same for every
// candidate and are left out, so OPD_F_GRADW_BF16 gets the same super-tiles as the fp32-grad_W call:
//   T >= 32768: the widest of 16384 / 12288 / 8192 / 4096 columns that fits, two G buffers (wider = fewer fp32 partial-sum passes:
//               C4 8192 columns, 2.5% faster than 4096; C5 16384 columns, 2.6% faster than 8192);
//   smaller T:  4096 columns and THREE G buffers (no wait at the block boundaries: C3 +2%, C2 +4%) if that fits, else
//               2048 columns x 3 buffers for tiny problems, else 4096 x 2.
// OPD_VB / OPD_G_BUFS override the choice (tuning, tests).
inline Plan make_plan(int T, int d, int V, int C, int fp32, unsigned flags, int mode = 1) {
    const int vb_env = env_int("OPD_VB", 0), gb_env = env_int("OPD_G_BUFS", 0);
    auto plan = [&](int vb, int gb) { return make_plan_cfg(T, d, V, C, fp32, flags, mode, vb_env > 0 ? vb_env : vb, gb_env > 0 ? gb_env : gb); };
    const double logits = 2.0 * (double)T * (double)V;
    const double budget = 0.048 * logits;
    const int t_pad = ceil_div(T, BM * cta_group_setting()) * BM * cta_group_setting();
    if (t_pad >= 32768) {
        for (int vb : {16384, 12288, 8192}) {
            const Plan p = plan(vb, 2);
            if ((double)(p.total - p.dv_bytes) <= budget) return p;
        }
        return plan(4096, 2);
    }
    const Plan p3 = plan(4096, 3);
    if ((double)(p3.total - p3.dv_bytes) <= budget) return p3;
    if (logits < 1e9) return plan(2048, 3);
    return plan(4096, 2);
}

// ---------------------------------------------------------------- GEMM launcher
// Launch `kernel` on `grid` CTAs of `threads` threads; CG = 2 launches clusters of two CTAs (a pair per tile).
// `window` (optional): an L2 access-policy window for this launch only (persisting hits inside [base, base + bytes)).
struct L2Window { void* base = nullptr; size_t bytes = 0; float hit_ratio = 1.f; };
template <int CG, int ST, class... KArgs, class... Args>
inline cudaError_t launch_cg_w(void (*kernel)(KArgs...), int grid, int threads, cudaStream_t st, const L2Window& window, Args&&... args) {
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg<CG, ST>::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = Cfg<CG, ST>::SMEM_BYTES; cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CG; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (window.base && window.bytes) {
        attr[1].id = cudaLaunchAttributeAccessPolicyWindow;
        attr[1].val.accessPolicyWindow.base_ptr = window.base;
        attr[1].val.accessPolicyWindow.num_bytes = window.bytes;
        attr[1].val.accessPolicyWindow.hitRatio = window.hit_ratio;
        attr[1].val.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
        attr[1].val.accessPolicyWindow.missProp = cudaAccessPropertyNormal;
        cfg.numAttrs = 2;
    }
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}
template <int CG, int ST, class... KArgs, class... Args>
inline cudaError_t launch_cg(void (*kernel)(KArgs...), int grid, cudaStream_t st, Args&&... args) {
    return launch_cg_w<CG, ST>(kernel, grid, GEMM_THREADS, st, L2Window{}, std::forward<Args>(args)...);
}

// Number of clusters (CG = 2) / CTAs (CG = 1) of `kernel` that can be resident at the same time on the current device:
// the persistent kernels size their grid with it (one wave; more CTAs would only queue behind the resident ones).
template <int CG, int ST, class... KArgs>
inline int max_resident_groups(void (*kernel)(KArgs...), int num_sms, int threads) {
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg<CG, ST>::SMEM_BYTES) != cudaSuccess) return 0;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(num_sms / CG * CG); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = Cfg<CG, ST>::SMEM_BYTES;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CG; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, kernel, &cfg) != cudaSuccess) { cudaGetLastError(); return 0; }
    return std::min(n, num_sms / CG);
}

template <class Epi, int CG>
inline cudaError_t launch_gemm_cg(opd_handle_s* h, cudaStream_t st, const CUtensorMap& tA, const CUtensorMap& tB,
                                  const GemmParams& gp, const typename Epi::Params& ep) {
    const long tiles = (long)ceil_div(gp.M, BM * CG) * gp.num_n;
    const int grid = CG * (int)std::min<long>(tiles, h->num_sms / CG);
    if (grid <= 0) return cudaSuccess;
    cudaError_t e = launch_cg<CG, fwd_stages<CG>()>(gemm_kernel<Epi, CG>, grid, st, tA, tB, gp, ep);
    h->n_kernels++;
    h->n_gemm++;
    return e != cudaSuccess ? e : cudaGetLastError();
}
template <class Epi>
inline cudaError_t launch_gemm(opd_handle_s* h, cudaStream_t st, const CUtensorMap& tA, const CUtensorMap& tB,
                               const GemmParams& gp, const typename Epi::Params& ep) {
    return h->cg == 2 ? launch_gemm_cg<Epi, 2>(h, st, tA, tB, gp, ep) : launch_gemm_cg<Epi, 1>(h, st, tA, tB, gp, ep);
}

inline void set_segments(GemmParams& gp, int planes) {
    if (planes == 1) { gp.nseg = 1; gp.sa[0] = 0; gp.sb[0] = 0; return; }
    // x = x0+x1+x2, w = w0+w1+w2 (bf16 terms): keep all products down to 2^-16 relative.  Smallest products first: the
    // tensor core adds into the fp32 accumulator with truncation, so each of the K/16 steps costs up to an ulp of the
    // accumulator's CURRENT magnitude; with x0.w0 last the five correction segments run while it is 2^-8 of its final size
    // (measured on logits of magnitude 30: error 9e-5 with x0.w0 first, as small as the one-segment bf16 path with it last)
    static const unsigned char pa[6] = {1, 2, 0, 1, 0, 0}, pb[6] = {1, 0, 2, 0, 1, 0};
    gp.nseg = 6;
    for (int i = 0; i < 6; ++i) { gp.sa[i] = pa[i]; gp.sb[i] = pb[i]; }
}

}  // namespace opd

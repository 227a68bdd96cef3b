// One persistent kernel for the whole backward (S6-S8).  Same warp-specialised tcgen05 pipeline as
// gemm_kernel, but the tile list interleaves three GEMM kinds over all (token x vocabulary) super-tiles:
//
//   block 0: G(0)      block b: G(b), DX(b-1), DW(b-1)      block S: DX(S-1), DW(S-1)
//
//   G(s)   logits of super-tile s recomputed -> G tile (bf16) into buffer s%2 of the L2-resident G ring
//   DX(s)  grad_hidden[tb] (+)= G(s) . W[:,vb]^T        DW(s)  grad_W[:,vb] += Xc[tb]^T . G(s)
//
// CTAs take items round-robin in list order; an item only depends on earlier items, through two counters
// per super-tile in global memory (release by the epilogue after its stores, acquire by whoever consumes):
//   g_done[s] == #G tiles      before the TMA producer loads G(s) for a DX/DW tile
//   c_done[s-1] complete       before a DX/DW(s) epilogue touches the fp32 accumulators (previous writer)
//   c_done[s-2] complete       before a G(s) epilogue overwrites ring buffer s%2 (previous readers)
// This removes the ~900 launches, their partial last waves and the pipeline refill of the per-GEMM version.
#pragma once
#include "opd_epilogues_bwd.cuh"

namespace opd {

struct BwdParams {
    int d, V, Tb, Vb, nvb;     // super-tile rows / cols, vocabulary super-tiles per token super-tile
    int wl;                    // 0: W is [d,V] row-major, 1: [V,d]
    int planes;                // 1 (bf16) or 3 (fp32 inputs as three bf16 terms)
    const int* n_live;
    int* g_done;               // [S]
    int* c_done;               // [S]
    GEpi::Params g;            // gs points at ring buffer 0; buffer b at + b * planes * plane_stride
    DxEpi::Params dx;
    DwEpi::Params dw;
};

enum { T_G = 0, T_DX = 1, T_DW = 2 };

struct BwdTile {
    int type, s, tb0, vb0, Tb_eff, Vb_eff, vi, m_blk, n_blk;
};

struct BwdSched {
    int S, nvb, Tb, Vb, V, d, wl, n_live;
    int blk;        // current block
    long base;      // items before the current block
    __device__ __forceinline__ void init(const BwdParams& p) {
        n_live = *p.n_live;
        nvb = p.nvb; Tb = p.Tb; Vb = p.Vb; V = p.V; d = p.d; wl = p.wl;
        S = ((n_live + Tb - 1) / Tb) * nvb;
        blk = 0; base = 0;
    }
    __device__ __forceinline__ void dims(int s, int& mt, int& nt, int& tb_eff, int& vb_eff) const {
        const int ti = s / nvb, vi = s - ti * nvb;
        tb_eff = min(Tb, n_live - ti * Tb);
        vb_eff = min(Vb, V - vi * Vb);
        mt = (tb_eff + BM - 1) / BM;
        nt = (vb_eff + BN - 1) / BN;
    }
    __device__ __forceinline__ int nG(int s) const { int mt, nt, a, b; dims(s, mt, nt, a, b); return mt * nt; }
    __device__ __forceinline__ int nDX(int s) const { int mt, nt, a, b; dims(s, mt, nt, a, b); return mt * ((d + BN - 1) / BN); }
    __device__ __forceinline__ int nDW(int s) const {
        int mt, nt, a, b; dims(s, mt, nt, a, b);
        return wl == 0 ? ((d + BM - 1) / BM) * nt : ((b + BM - 1) / BM) * ((d + BN - 1) / BN);
    }
    __device__ __forceinline__ int block_size(int b) const {
        return (b < S ? nG(b) : 0) + (b >= 1 ? nDX(b - 1) + nDW(b - 1) : 0);
    }
    // decode `item` (monotonically increasing between calls); false when the list is exhausted
    __device__ __forceinline__ bool get(long item, BwdTile& t) {
        while (blk <= S) {
            const int sz = block_size(blk);
            if (item < base + sz) break;
            base += sz; ++blk;
        }
        if (blk > S) return false;
        int r = static_cast<int>(item - base);
        int rows;
        if (blk < S && r < nG(blk)) { t.type = T_G; t.s = blk; }
        else {
            if (blk < S) r -= nG(blk);
            t.s = blk - 1;
            const int ndx = nDX(t.s);
            if (r < ndx) t.type = T_DX; else { t.type = T_DW; r -= ndx; }
        }
        int mt, nt;
        dims(t.s, mt, nt, t.Tb_eff, t.Vb_eff);
        const int ti = t.s / nvb;
        t.vi = t.s - ti * nvb;
        t.tb0 = ti * Tb; t.vb0 = t.vi * Vb;
        if (t.type == T_DW) rows = wl == 0 ? (d + BM - 1) / BM : (t.Vb_eff + BM - 1) / BM;
        else rows = mt;
        t.m_blk = r % rows; t.n_blk = r / rows;     // m fastest: concurrently running CTAs share the B panel
        return true;
    }
};

__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void wait_counter(const int* c, int expected) {
    while (ld_acquire_gpu(c) < expected) __nanosleep(128);
}
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }

__global__ void __launch_bounds__(GEMM_THREADS, 1)
bwd_kernel(const __grid_constant__ CUtensorMap m_xc_k, const __grid_constant__ CUtensorMap m_w_fwd,
           const __grid_constant__ CUtensorMap m_gs_k, const __grid_constant__ CUtensorMap m_w_dx,
           const __grid_constant__ CUtensorMap m_xc_mn, const __grid_constant__ CUtensorMap m_gs_mn,
           const __grid_constant__ BwdParams bp) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + STAGES * STAGE_BYTES);
    uint64_t* empty_bar = full_bar + STAGES;
    uint64_t* tfull_bar = empty_bar + STAGES;
    uint64_t* tempty_bar = tfull_bar + 2;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty_bar + 2);
    uint8_t* epi_smem = smem + STAGES * STAGE_BYTES + 1024;

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    if (*bp.n_live <= 0) return;

    if (warp == 0 && lane == 0) {
        prefetch_tmap(&m_xc_k); prefetch_tmap(&m_w_fwd); prefetch_tmap(&m_gs_k);
        prefetch_tmap(&m_w_dx); prefetch_tmap(&m_xc_mn); prefetch_tmap(&m_gs_mn);
        for (int s = 0; s < STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(&tfull_bar[s], 1); mbar_init(&tempty_bar[s], 4); }
        fence_mbar_init();
    }
    if (warp == 1) { tmem_alloc(tmem_slot, TMEM_COLS); tmem_relinquish(); }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    // segment tables of the three-term split (planes == 3), see set_segments()
    const int nseg = bp.planes == 1 ? 1 : 6;
    const int PA[6] = {0, 0, 1, 0, 2, 1};
    const int PB[6] = {0, 1, 0, 2, 0, 1};

    if (warp == 0) {
        // =========================== TMA producer ===========================
        if (elect_one()) {
            BwdSched sc; sc.init(bp);
            BwdTile t;
            int it = 0;
            for (long item = blockIdx.x; sc.get(item, t); item += gridDim.x) {
                const CUtensorMap *tA, *tB;
                int a_mn, b_mn, a_c, b_c, ka, kb, K, pa_off = 0, pb_off = 0;
                const int buf = t.s & 1;
                if (t.type == T_G) {
                    tA = &m_xc_k; tB = &m_w_fwd; a_mn = 0; b_mn = (bp.wl == 0);
                    a_c = t.tb0 + t.m_blk * BM; b_c = t.vb0 + t.n_blk * BN; ka = 0; kb = 0; K = bp.d;
                } else if (t.type == T_DX) {
                    tA = &m_gs_k; tB = &m_w_dx; a_mn = 0; b_mn = (bp.wl == 1);
                    a_c = t.m_blk * BM; b_c = t.n_blk * BN; ka = 0; kb = t.vb0; K = t.Vb_eff; pa_off = buf * bp.planes;
                } else if (bp.wl == 0) {
                    tA = &m_xc_mn; tB = &m_gs_mn; a_mn = 1; b_mn = 1;
                    a_c = t.m_blk * BM; b_c = t.n_blk * BN; ka = t.tb0; kb = 0; K = t.Tb_eff; pb_off = buf * bp.planes;
                } else {
                    tA = &m_gs_mn; tB = &m_xc_mn; a_mn = 1; b_mn = 1;
                    a_c = t.m_blk * BM; b_c = t.n_blk * BN; ka = 0; kb = t.tb0; K = t.Tb_eff; pa_off = buf * bp.planes;
                }
                if (t.type != T_G) {                        // the G super-tile must be complete before TMA reads it
                    wait_counter(bp.g_done + t.s, sc.nG(t.s));
                    fence_proxy_async_all();
                }
                const int kblocks = (K + BK - 1) / BK;
                for (int seg = 0; seg < nseg; ++seg) {
                    const int pa = pa_off + (nseg == 1 ? 0 : PA[seg]), pb = pb_off + (nseg == 1 ? 0 : PB[seg]);
                    for (int kb_i = 0; kb_i < kblocks; ++kb_i, ++it) {
                        const int s = it % STAGES;
                        const uint32_t ph = (it / STAGES) & 1;
                        mbar_wait(&empty_bar[s], ph ^ 1);
                        uint8_t* sA = smem + s * STAGE_BYTES;
                        uint8_t* sB = sA + A_STAGE_BYTES;
                        mbar_arrive_expect_tx(&full_bar[s], STAGE_BYTES);
                        const int kca = ka + kb_i * BK, kcb = kb + kb_i * BK;
                        if (a_mn) {
                            for (int b = 0; b < BM / MN_BOX; ++b)
                                tma_load_3d(sA + b * MN_BOX_BYTES, tA, &full_bar[s], a_c + b * MN_BOX, kca, pa);
                        } else {
                            tma_load_3d(sA, tA, &full_bar[s], kca, a_c, pa);
                        }
                        if (b_mn) {
                            for (int b = 0; b < BN / MN_BOX; ++b)
                                tma_load_3d(sB + b * MN_BOX_BYTES, tB, &full_bar[s], b_c + b * MN_BOX, kcb, pb);
                        } else {
                            tma_load_3d(sB, tB, &full_bar[s], kcb, b_c, pb);
                        }
                    }
                }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer ===========================
        if (elect_one()) {
            BwdSched sc; sc.init(bp);
            BwdTile t;
            int it = 0, lt = 0;
            for (long item = blockIdx.x; sc.get(item, t); item += gridDim.x, ++lt) {
                int a_mn, b_mn, K;
                if (t.type == T_G) { a_mn = 0; b_mn = (bp.wl == 0); K = bp.d; }
                else if (t.type == T_DX) { a_mn = 0; b_mn = (bp.wl == 1); K = t.Vb_eff; }
                else { a_mn = 1; b_mn = 1; K = t.Tb_eff; }
                const uint32_t idesc = make_idesc_bf16(BM, BN, a_mn, b_mn);
                const uint32_t a_kstep = a_mn ? (UMMA_K * MN_BOX * 2) : (UMMA_K * 2);
                const uint32_t b_kstep = b_mn ? (UMMA_K * MN_BOX * 2) : (UMMA_K * 2);
                const uint32_t a_lbo = a_mn ? MN_BOX_BYTES : 16;
                const uint32_t b_lbo = b_mn ? MN_BOX_BYTES : 16;
                const int kiters = ((K + BK - 1) / BK) * nseg;
                const int as = lt & 1;
                const uint32_t aph = (lt >> 1) & 1;
                mbar_wait(&tempty_bar[as], aph ^ 1);
                tc_fence_after();
                const uint32_t tacc = tmem_base + as * BN;
                for (int ki = 0; ki < kiters; ++ki, ++it) {
                    const int s = it % STAGES;
                    const uint32_t ph = (it / STAGES) & 1;
                    mbar_wait(&full_bar[s], ph);
                    tc_fence_after();
                    const uint32_t a0 = smem_u32(smem + s * STAGE_BYTES);
                    const uint32_t b0 = a0 + A_STAGE_BYTES;
#pragma unroll
                    for (int k = 0; k < BK / UMMA_K; ++k) {
                        const uint64_t ad = make_smem_desc(a0 + k * a_kstep, a_lbo, 1024);
                        const uint64_t bd = make_smem_desc(b0 + k * b_kstep, b_lbo, 1024);
                        umma_bf16(tacc, ad, bd, idesc, (ki | k) != 0);
                    }
                    umma_commit(&empty_bar[s]);
                }
                umma_commit(&tfull_bar[as]);
            }
        }
    } else {
        // =========================== epilogue warps ===========================
        const int quarter = warp & 3;
        const int row_in_tile = quarter * 32 + lane;
        const int epi_tid = (warp - 2) * 32 + lane;
        BwdSched sc; sc.init(bp);
        BwdTile t;
        int lt = 0;
        for (long item = blockIdx.x; sc.get(item, t); item += gridDim.x, ++lt) {
            const int as = lt & 1;
            const uint32_t aph = (lt >> 1) & 1;
            const uint32_t taddr = tmem_base + as * BN + (static_cast<uint32_t>(quarter * 32) << 16);
            GemmParams gp{};                      // the fields the epilogues read
            gp.tok_off = t.tb0;
            // wait for the previous writer / readers of what this epilogue is about to write
            const int dep = (t.type == T_G) ? t.s - 2 : t.s - 1;
            if (dep >= 0) {
                if (lane == 0) { wait_counter(bp.c_done + dep, sc.nDX(dep) + sc.nDW(dep)); fence_proxy_async_all(); }
                __syncwarp();
            }
            if (t.type == T_G) {
                gp.b_off = t.vb0; gp.N = t.Vb_eff;
                GEpi::Params ep = bp.g;
                ep.gs += static_cast<size_t>(t.s & 1) * bp.planes * ep.plane_stride;
                GEpi::State st = GEpi::prepare(ep, gp, t.m_blk, t.n_blk, row_in_tile, t.Tb_eff);
                mbar_wait(&tfull_bar[as], aph);
                tc_fence_after();
                GEpi::run(ep, gp, st, taddr, t.m_blk, t.n_blk, row_in_tile, t.Tb_eff, nullptr, epi_tid);
            } else if (t.type == T_DX) {
                gp.N = bp.d; gp.first = (t.vi == 0); gp.last = (t.vi == bp.nvb - 1);
                DxEpi::State st = DxEpi::prepare(bp.dx, gp, t.m_blk, t.n_blk, row_in_tile, t.Tb_eff);
                mbar_wait(&tfull_bar[as], aph);
                tc_fence_after();
                DxEpi::run(bp.dx, gp, st, taddr, t.m_blk, t.n_blk, row_in_tile, t.Tb_eff, epi_smem, epi_tid);
            } else {
                int M_eff;
                if (bp.wl == 0) { gp.N = t.Vb_eff; gp.row_off = 0; gp.col_off = t.vb0; M_eff = bp.d; }
                else { gp.N = bp.d; gp.row_off = t.vb0; gp.col_off = 0; M_eff = t.Vb_eff; }
                mbar_wait(&tfull_bar[as], aph);
                tc_fence_after();
                DwEpi::run(bp.dw, gp, NoState{}, taddr, t.m_blk, t.n_blk, row_in_tile, M_eff, epi_smem, epi_tid);
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&tempty_bar[as]);           // TMEM stage free for the MMA warp
            // publish: all 128 epilogue threads' global stores, then one release increment
            __threadfence();
            fence_proxy_async_all();
            asm volatile("bar.sync 1, 128;" ::: "memory");
            if (epi_tid == 0) atomicAdd((t.type == T_G ? bp.g_done : bp.c_done) + t.s, 1);
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, TMEM_COLS);
}

}  // namespace opd

// Generic persistent warp-specialised GEMM core for sm_100a:  D[M,N] = sum_seg A_seg[M,K] * B_seg[N,K]^T
//   TMA (SWIZZLE_128B) -> 4-stage smem ring -> tcgen05.mma (cta_group::1, 128x256x16, bf16 -> fp32)
//   -> double-buffered TMEM accumulators -> per-tile epilogue functor run by 4 epilogue warps.
// A and B may each be K-major (K contiguous in global memory) or MN-major (M/N contiguous); the
// majorness is a run-time parameter that only changes the TMA box sequence and the UMMA descriptors.
// Every GEMM of the OPD path (logits, G re-formation, grad_hidden, grad_W) is this kernel with a
// different epilogue (see opd_epilogues.cuh).
#pragma once
#include "opd_ptx.cuh"

namespace opd {

constexpr int BM = 128;              // tile rows   (TMEM lanes)
constexpr int BN = 256;              // tile cols   (TMEM columns, fp32)
constexpr int BK = 64;               // bf16 elements per k-block = one 128-byte swizzle row
constexpr int UMMA_K = 16;
constexpr int STAGES = 4;
constexpr int A_STAGE_BYTES = BM * BK * 2;            // 16 KiB
constexpr int B_STAGE_BYTES = BN * BK * 2;            // 32 KiB
constexpr int STAGE_BYTES = A_STAGE_BYTES + B_STAGE_BYTES;
constexpr int MN_BOX = 64;                            // MN-major operands arrive as 64(mn) x 64(k) boxes
constexpr int MN_BOX_BYTES = MN_BOX * BK * 2;         // 8 KiB
constexpr int GEMM_THREADS = 192;                     // warp0 TMA, warp1 MMA(+TMEM alloc), warps2-5 epilogue
constexpr int EPI_SMEM_BYTES = 32768;                 // 4 epilogue warps x 2 staging buffers x (32 rows x 128 B)
constexpr int GEMM_SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*barriers*/ + EPI_SMEM_BYTES + 1024 /*align slack*/;
constexpr int TMEM_COLS = 512;                        // 2 accumulator stages x 256 columns

enum TokDim { TOK_NONE = 0, TOK_M = 1, TOK_K = 2 };
constexpr int MAX_SEG = 6;

struct GemmParams {
    int M, N, K;              // extents of this GEMM (upper bounds; the token extent is clipped on the device)
    int num_n;                // ceil(N / BN)
    int group_m;              // raster: tiles are walked in groups of group_m row-tiles, m fastest inside
    int a_mn, b_mn;           // 1 = MN-major operand (M/N contiguous in memory), 0 = K-major
    int a_off, b_off;         // M / N element offsets of this GEMM inside the tensors the TMA maps describe
    int ka_off, kb_off;       // K element offsets inside A's and B's tensor
    int nseg;                 // K segments (1 for bf16; 6 for the 3-way bf16 split of fp32 operands)
    unsigned char sa[MAX_SEG], sb[MAX_SEG];   // plane (3rd TMA coordinate) of A / B per segment
    int tok_dim;              // which extent counts live tokens (clipped to n_live - tok_off on the device)
    int tok_off;
    const int* n_live;        // device scalar: number of live tokens (compacted rows)
    // per-launch / per-tile epilogue switches (set by the host for gemm_kernel, per tile by bwd_kernel)
    int first, last;          // DxEpi: first / last vocabulary super-tile of this token super-tile
    int row_off, col_off;     // DwEpi: position of this GEMM's output inside grad_W
};

__device__ __forceinline__ void tile_coords(int tile, int num_m, int num_n, int group_m, int& m_blk, int& n_blk) {
    const int per_group = group_m * num_n;
    const int g = tile / per_group;
    const int r = tile - g * per_group;
    const int m0 = g * group_m;
    const int gm = min(group_m, num_m - m0);
    m_blk = m0 + r % gm;
    n_blk = r / gm;
}

// Epi must provide:  struct Params;  static __device__ void run(const Params&, const GemmParams&, uint32_t taddr,
//                    int m_blk, int n_blk, int row_in_tile, int M_eff, uint8_t* epi_smem, int epi_tid)
template <class Epi>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
            const GemmParams gp, const __grid_constant__ typename Epi::Params ep) {
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

    // ---- device-side extents (the live-token count is only known on the device)
    int M = gp.M, K = gp.K;
    if (gp.tok_dim != TOK_NONE) {
        const int live = *gp.n_live - gp.tok_off;
        if (gp.tok_dim == TOK_M) M = min(M, live);
        else K = min(K, live);
    }
    if (M <= 0 || K <= 0) return;
    const int num_m = (M + BM - 1) / BM;
    const int num_n = gp.num_n;
    const int total_tiles = num_m * num_n;
    const int kblocks = (K + BK - 1) / BK;
    const int kiters = kblocks * gp.nseg;

    if (warp == 0 && lane == 0) {
        prefetch_tmap(&tmA);
        prefetch_tmap(&tmB);
        for (int s = 0; s < STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(&tfull_bar[s], 1); mbar_init(&tempty_bar[s], 4); }
        fence_mbar_init();
    }
    if (warp == 1) {
        tmem_alloc(tmem_slot, TMEM_COLS);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // =========================== TMA producer (one elected lane) ===========================
        if (elect_one()) {
            int it = 0;
            for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
                int m_blk, n_blk;
                tile_coords(tile, num_m, num_n, gp.group_m, m_blk, n_blk);
                const int a_mn0 = gp.a_off + m_blk * BM;
                const int b_mn0 = gp.b_off + n_blk * BN;
                for (int ki = 0; ki < kiters; ++ki, ++it) {
                    const int s = it % STAGES;
                    const uint32_t ph = (it / STAGES) & 1;
                    mbar_wait(&empty_bar[s], ph ^ 1);
                    const int seg = ki / kblocks;
                    const int kk = (ki - seg * kblocks) * BK;
                    const int kca = gp.ka_off + kk, kcb = gp.kb_off + kk;
                    uint8_t* sA = smem + s * STAGE_BYTES;
                    uint8_t* sB = sA + A_STAGE_BYTES;
                    mbar_arrive_expect_tx(&full_bar[s], STAGE_BYTES);
                    if (gp.a_mn) {
                        for (int b = 0; b < BM / MN_BOX; ++b)
                            tma_load_3d(sA + b * MN_BOX_BYTES, &tmA, &full_bar[s], a_mn0 + b * MN_BOX, kca, gp.sa[seg]);
                    } else {
                        tma_load_3d(sA, &tmA, &full_bar[s], kca, a_mn0, gp.sa[seg]);
                    }
                    if (gp.b_mn) {
                        for (int b = 0; b < BN / MN_BOX; ++b)
                            tma_load_3d(sB + b * MN_BOX_BYTES, &tmB, &full_bar[s], b_mn0 + b * MN_BOX, kcb, gp.sb[seg]);
                    } else {
                        tma_load_3d(sB, &tmB, &full_bar[s], kcb, b_mn0, gp.sb[seg]);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer (one elected lane) ===========================
        if (elect_one()) {
            const uint32_t idesc = make_idesc_bf16(BM, BN, gp.a_mn, gp.b_mn);
            const uint32_t a_kstep = gp.a_mn ? (UMMA_K * MN_BOX * 2) : (UMMA_K * 2);   // bytes per UMMA_K step
            const uint32_t b_kstep = gp.b_mn ? (UMMA_K * MN_BOX * 2) : (UMMA_K * 2);
            const uint32_t a_lbo = gp.a_mn ? MN_BOX_BYTES : 16;
            const uint32_t b_lbo = gp.b_mn ? MN_BOX_BYTES : 16;
            int it = 0, lt = 0;
            for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x, ++lt) {
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
                    umma_commit(&empty_bar[s]);          // frees the smem slot once these MMAs have read it
                }
                umma_commit(&tfull_bar[as]);             // accumulator complete -> epilogue
            }
        }
    } else {
        // =========================== epilogue warps (TMEM -> registers -> global) ===========================
        const int quarter = warp & 3;                    // TMEM lane quarter this warp may access
        const int row_in_tile = quarter * 32 + lane;
        const int epi_tid = (warp - 2) * 32 + lane;
        int lt = 0;
        for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x, ++lt) {
            int m_blk, n_blk;
            tile_coords(tile, num_m, num_n, gp.group_m, m_blk, n_blk);
            const int as = lt & 1;
            const uint32_t aph = (lt >> 1) & 1;
            // per-row state (scalars, cache cursor) is fetched while the MMAs of this tile are still running
            typename Epi::State st = Epi::prepare(ep, gp, m_blk, n_blk, row_in_tile, M);
            mbar_wait(&tfull_bar[as], aph);
            tc_fence_after();
            const uint32_t taddr = tmem_base + as * BN + (static_cast<uint32_t>(quarter * 32) << 16);
            Epi::run(ep, gp, st, taddr, m_blk, n_blk, row_in_tile, M, epi_smem, epi_tid);
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&tempty_bar[as]);
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, TMEM_COLS);
}

}  // namespace opd

// Backward epilogues (S6-S8), see opd_epilogues.cuh for the conventions.
#pragma once
#include "opd_epilogues.cuh"

namespace opd {

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
    __nv_bfloat162 t = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&t);
}

// ------------------------------------------------------------------------------------------ GEpi
// S6: re-form G[t,v] = coef_t * exp(z[t,v] - lse_t) + sum_j beta_tj [a_tj == v]  with coef = alpha/N,
// beta pre-scaled by 1/N (derivation: DESIGN.md "Backward"), round to bf16 and store it into the
// super-tile Gs[Tb][ldg] (row-major, v contiguous) that the dX and dW contractions read back from L2.
// Rows past the live count and columns past V are written as zeros: both contractions rely on it.
struct GEpi {
    struct Params {
        __nv_bfloat16* gs;       // [planes][rows][ldg]
        int rows;                // allocated rows per plane (tile rows past it are not stored)
        long ldg;
        long plane_stride;       // elements
        int planes;              // 1 (bf16 path) or 3 (fp32 path: three-term bf16 split of G)
        const float* lse2;       // [T] lse * log2(e), compact row order
        const float* coef;       // [T] alpha_t / N
        const int* sorted_idx;   // [T][C]
        const float* beta;       // [T][C] beta_tj / N in sorted-slot order
        int C;
        int V;
        unsigned long long st_hint;   // L2 eviction policy of the G stores (0 = plain stores)
    };
    struct State { int cursor; int next_col; float lse2; float coef; };
    static __device__ __forceinline__ State prepare(const Params& p, const GemmParams& gp, int m_blk, int n_blk,
                                                    int row_in_tile, int M_eff) {
        State st{p.C, IDX_SENTINEL, 0.f, 0.f};
        const int lrow = m_blk * BM + row_in_tile;
        if (lrow < M_eff) {
            const int row = gp.tok_off + lrow;
            const int* idx = p.sorted_idx + static_cast<size_t>(row) * p.C;
            st.cursor = lower_bound_slot(idx, p.C, gp.b_off + n_blk * BN);
            st.next_col = st.cursor < p.C ? __ldg(idx + st.cursor) : IDX_SENTINEL;
            st.lse2 = p.lse2[row];
            st.coef = p.coef[row];
        }
        return st;
    }
    static __device__ __forceinline__ void run(const Params& p, const GemmParams& gp, State st, uint32_t taddr,
                                               int m_blk, int n_blk, int row_in_tile, int M_eff, uint8_t*, int) {
        const int lrow = m_blk * BM + row_in_tile;
        const bool live = lrow < M_eff;
        const int row = gp.tok_off + lrow;
        const int* idx = p.sorted_idx + static_cast<size_t>(row) * p.C;
        const float* beta = p.beta + static_cast<size_t>(row) * p.C;
        __nv_bfloat16* out = p.gs + static_cast<size_t>(lrow) * p.ldg + n_blk * BN;
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
            float v[32];
            tmem_ld32(taddr + c * 32, v);
            tmem_ld_wait();
            const int col0 = gp.b_off + n_blk * BN + c * 32;          // vocabulary column of v[0]
            if (live) {
#pragma unroll
                for (int i = 0; i < 32; ++i) v[i] = st.coef * exp2f(fmaf(v[i], LOG2E, -st.lse2));
            } else {
#pragma unroll
                for (int i = 0; i < 32; ++i) v[i] = 0.f;
            }
            if (__any_sync(0xffffffffu, st.next_col < col0 + 32)) {
                while (st.next_col < col0 + 32) {                    // duplicates add up
                    add_at32(v, st.next_col - col0, __ldg(beta + st.cursor));
                    ++st.cursor;
                    st.next_col = st.cursor < p.C ? __ldg(idx + st.cursor) : IDX_SENTINEL;
                }
            }
            if (col0 + 32 > p.V) {
#pragma unroll
                for (int i = 0; i < 32; ++i)
                    if (col0 + i >= p.V) v[i] = 0.f;
            }
            if (lrow >= p.rows) continue;                             // row of a pair tile past the buffer
            for (int pl = 0; pl < p.planes; ++pl) {
                uint32_t w[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    w[i] = pack_bf16x2(v[2 * i], v[2 * i + 1]);
                    if (pl + 1 < p.planes) {                          // residual for the next split term
                        __nv_bfloat162 t = *reinterpret_cast<__nv_bfloat162*>(&w[i]);
                        v[2 * i] -= __low2float(t);
                        v[2 * i + 1] -= __high2float(t);
                    }
                }
                uint4* dst = reinterpret_cast<uint4*>(out + pl * p.plane_stride + c * 32);
                if (p.st_hint) {
#pragma unroll
                    for (int q = 0; q < 4; ++q) st_global_v4_hint(dst + q, w[4 * q], w[4 * q + 1], w[4 * q + 2], w[4 * q + 3], p.st_hint);
                } else {
#pragma unroll
                    for (int q = 0; q < 4; ++q) dst[q] = make_uint4(w[4 * q], w[4 * q + 1], w[4 * q + 2], w[4 * q + 3]);
                }
            }
        }
    }
};

// ------------------------------------------------------------------------------------------ fp32 accumulate via TMA
// One warp stages its 32 rows x 32 fp32 columns (128-byte rows, SWIZZLE_128B) into one of its two 4 KiB smem
// buffers and one lane issues a TMA store or reduce-add: the read-modify-write of the fp32 accumulators happens in
// L2, the epilogue never waits on a load.  `wbuf` is this warp's 8 KiB (1024-byte aligned) region.
__device__ __forceinline__ void stage_and_send(const CUtensorMap* tm, uint8_t* wbuf, int parity, const float (&v)[32],
                                               int lane, int col, int row, bool reduce, uint64_t hint) {
    uint8_t* buf = wbuf + parity * 4096;
    if (lane == 0) bulk_wait_read<1>();          // the group that last used this buffer has finished reading it
    __syncwarp();
    uint8_t* rowp = buf + lane * 128;
#pragma unroll
    for (int q = 0; q < 8; ++q)
        *reinterpret_cast<float4*>(rowp + ((q ^ (lane & 7)) << 4)) = make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
    fence_proxy_async_smem();
    __syncwarp();
    if (lane == 0) {
        if (reduce) tma_reduce_add_2d(tm, buf, col, row, hint); else tma_store_2d(tm, buf, col, row, hint);
        bulk_commit();
    }
}
// all bulk stores / reductions issued by this warp are complete (globally performed)
__device__ __forceinline__ void drain_sends(int lane) {
    if (lane == 0) bulk_wait<0>();
    __syncwarp();
}

// ------------------------------------------------------------------------------------------ DxEpi
// S7: grad_hidden super-tile [Tb][d] = sum over vocabulary super-tiles of  G . W^T.  Partial sums live in an
// fp32 workspace between super-tiles (TMA store for the first, TMA reduce-add after); the last one adds the
// workspace to its accumulator and emits rows into grad_hidden (dtype of hidden) at the token positions.
struct DxEpi {
    struct Params {
        CUtensorMap m_acc;       // fp32 [Tb_pad][d], boxes of 32 x 32
        uint64_t hint;           // L2 eviction policy of the partial-sum stores / reductions
#ifdef OPD_EXPERIMENTS
        int dbg;                 // timing experiments (wrong gradients): 1 = plain stores instead of reductions, 2 = no output
#endif
        float* acc;              // same buffer, for the last super-tile's read
        long ld_acc;
        void* out;               // grad_hidden
        long ld_out;
        int out_fp32;
        const int* live_rows;    // compact row -> token index
    };
    struct State { int tok; };
    static __device__ __forceinline__ State prepare(const Params& p, const GemmParams& gp, int m_blk, int,
                                                    int row_in_tile, int M_eff) {
        State st{-1};
        const int lrow = m_blk * BM + row_in_tile;
        if (gp.last && lrow < M_eff) st.tok = p.live_rows[gp.tok_off + lrow];
        return st;
    }
    static __device__ __forceinline__ void run(const Params& p, const GemmParams& gp, State st, uint32_t taddr,
                                               int m_blk, int n_blk, int row_in_tile, int M_eff, uint8_t* epi_smem, int epi_tid) {
        const int lrow = m_blk * BM + row_in_tile;
        const bool live = lrow < M_eff;
        const int lane = epi_tid & 31;
        uint8_t* wbuf = epi_smem + (epi_tid >> 5) * 8192;
        const float* acc = p.acc + static_cast<size_t>(lrow) * p.ld_acc + n_blk * BN;
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
            float v[32];
            tmem_ld32(taddr + c * 32, v);
            tmem_ld_wait();
            const int col0 = n_blk * BN + c * 32;
            if (col0 >= gp.N) break;                                  // d % 64 == 0: chunks are all-in or all-out (warp-uniform)
#ifdef OPD_EXPERIMENTS
            if (p.dbg == 2) continue;
            const bool reduce = !gp.first && p.dbg != 1;
#else
            const bool reduce = !gp.first;
#endif
            if (!gp.last) {
                stage_and_send(&p.m_acc, wbuf, c & 1, v, lane, col0, lrow - lane, reduce, p.hint);
            } else if (live) {
                if (!gp.first) {
                    const float4* a4 = reinterpret_cast<const float4*>(acc + c * 32);
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        const float4 o = __ldcg(a4 + q);              // written through L2 by other SMs: bypass L1
                        v[4 * q] += o.x; v[4 * q + 1] += o.y; v[4 * q + 2] += o.z; v[4 * q + 3] += o.w;
                    }
                }
                if (p.out_fp32) {
                    float4* o4 = reinterpret_cast<float4*>(static_cast<float*>(p.out) + static_cast<size_t>(st.tok) * p.ld_out + col0);
#pragma unroll
                    for (int q = 0; q < 8; ++q) o4[q] = make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
                } else {
                    uint4* o4 = reinterpret_cast<uint4*>(static_cast<__nv_bfloat16*>(p.out) + static_cast<size_t>(st.tok) * p.ld_out + col0);
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        o4[q] = make_uint4(pack_bf16x2(v[8 * q], v[8 * q + 1]), pack_bf16x2(v[8 * q + 2], v[8 * q + 3]),
                                           pack_bf16x2(v[8 * q + 4], v[8 * q + 5]), pack_bf16x2(v[8 * q + 6], v[8 * q + 7]));
                }
            }
        }
        if (!gp.last) drain_sends(lane);
    }
};

// ------------------------------------------------------------------------------------------ DwEpi
// S8: grad_W tile (+)= accumulator (TMA reduce-add; the tiles of the first token super-tile store instead unless the call
// accumulates into the caller's running sum, so grad_W needs no memset).  Output element
// (row, col) of this GEMM lives at row = row_off + tile row, col = col_off + tile col of the fp32 tensor the map
// describes ((d,V) or (V,d)); TMA clips rows / columns outside the tensor.
struct DwEpi {
    struct Params {
        CUtensorMap m_gw;        // fp32 [rows_total][cols_total] (row stride ld), boxes of 32 x 32
        uint64_t hint;           // L2 eviction policy of the grad_W reductions
#ifdef OPD_EXPERIMENTS
        int dbg;                 // timing experiments (wrong gradients): 1 = plain stores instead of reductions, 2 = no output
#endif
    };
    using State = NoState;
    static __device__ __forceinline__ State prepare(const Params&, const GemmParams&, int, int, int, int) { return {}; }
    static __device__ __forceinline__ void run(const Params& p, const GemmParams& gp, const State&, uint32_t taddr,
                                               int m_blk, int n_blk, int row_in_tile, int M_eff, uint8_t* epi_smem, int epi_tid) {
        const int lane = epi_tid & 31;
        uint8_t* wbuf = epi_smem + (epi_tid >> 5) * 8192;
        const int lrow0 = m_blk * BM + row_in_tile - lane;           // first tile row of this warp
        const bool warp_ok = lrow0 < M_eff;                          // extents are multiples of 32 except at tensor edges (clipped)
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
            float v[32];
            tmem_ld32(taddr + c * 32, v);
            tmem_ld_wait();
            const int lc0 = n_blk * BN + c * 32;
            if (lc0 >= gp.N) break;
#ifdef OPD_EXPERIMENTS
            if (p.dbg == 2) continue;
            const bool reduce = !gp.first && p.dbg != 1;
#else
            const bool reduce = !gp.first;      // first token super-tile of an overwriting call: plain store
#endif
            if (warp_ok) stage_and_send(&p.m_gw, wbuf, c & 1, v, lane, gp.col_off + lc0, gp.row_off + lrow0, reduce, p.hint);
        }
        drain_sends(lane);
    }
};

}  // namespace opd

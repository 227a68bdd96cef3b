// Backward epilogues (S6-S8), see opd_epilogues.cuh for the conventions.
#pragma once
#include "opd_epilogues.cuh"

namespace opd {

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
    __nv_bfloat162 t = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&t);
}

// Software-pipelined walk over a tile's accumulator: the TMEM load of chunk c + 1 (32 fp32 columns of this thread's row) is
// in flight while body(v, c) works on chunk c.  TMEM reads run at 64 B per cycle and SM (B300_MICROARCH.md: 4 KiB per
// warp-wide tcgen05.ld), so a load that is waited for at once costs every chunk 60-250 cycles of idle epilogue warp.
// nchunks is warp-uniform; every load issued has been waited for when this returns.
template <class F>
__device__ __forceinline__ void for_each_chunk(uint32_t taddr, int nchunks, F&& body, long long* tr = nullptr) {
    float va[32], vb[32];
    if (nchunks <= 0) return;
    tmem_ld32(taddr, va);
#ifdef OPD_TRACE
    long long t0 = clock64(), t1;
#define OPD_TR_STEP(slot) if (tr) { t1 = clock64(); tr[slot] += t1 - t0; t0 = t1; }
#else
#define OPD_TR_STEP(slot)
#endif
#pragma unroll 1
    for (int c = 0; c < nchunks; c += 2) {
        tmem_ld_wait_for(va);
        if (c + 1 < nchunks) tmem_ld32(taddr + (c + 1) * 32, vb);
        OPD_TR_STEP(6)
        body(va, c);
        OPD_TR_STEP(7)
        if (c + 1 < nchunks) {
            tmem_ld_wait_for(vb);
            if (c + 2 < nchunks) tmem_ld32(taddr + (c + 2) * 32, va);
            OPD_TR_STEP(6)
            body(vb, c + 1);
            OPD_TR_STEP(7)
        }
    }
#undef OPD_TR_STEP
}

// ------------------------------------------------------------------------------------------ GEpi
// S6: re-form G[t,v] = coef_t * exp(z[t,v] - lse_t) + sum_j beta_tj [a_tj == v]  with coef = alpha/N,
// beta pre-scaled by 1/N (derivation: DESIGN.md "Backward"), round to bf16 and store it into the
// super-tile Gs[Tb][ldg] (row-major, v contiguous) that the dX and dW contractions read back from L2.
// Rows past the live count and columns past V are written as zeros: both contractions rely on it.
// Per element: one FFMA and one MUFU.EX2 -- the coefficient is folded into the exponent,
//     coef * 2^(z log2e - lse2) = sign(coef) * 2^(z log2e - (lse2 - log2|coef|)),
// its sign is an XOR on the packed bf16 pair (beta is added in the sign-folded domain), coef = 0 and dead rows give
// 2^-inf = +0 without a branch.  Each thread stores its row's 64 bytes per chunk as two 32-byte stores (whole sectors).
// These row-per-thread stores are what bounds this epilogue (one LSU wavefront per sector, about 4000 cycles per tile);
// staging the tile through shared memory for TMA stores has a quarter of the wavefronts but puts the completion wait of the
// last store on every tile and measured no faster (profiles/r02_trace.md).
// The cached columns of the row are found in prepare() with one pass of vector loads and the next two are kept in
// registers, so that a hit inside a chunk costs no memory latency.
struct GEpi {
    struct Params {
        __nv_bfloat16* gs;       // ring buffer 0: [planes][rows][ldg]
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
        unsigned long long st_hint;   // L2 eviction policy of the G stores (0 = normal)
    };
    // next_col / beta_a: the row's next cached column at or after this tile and its coefficient; col_b / beta_b: the one after
    struct State { int cursor; int next_col; int col_b; float beta_a; float beta_b; float off; uint32_t sgn; };
    static __device__ __forceinline__ State prepare(const Params& p, const GemmParams& gp, int m_blk, int n_blk,
                                                    int row_in_tile, int M_eff) {
        State st{p.C, IDX_SENTINEL, IDX_SENTINEL, 0.f, 0.f, INFINITY, 0u};
        const int lrow = m_blk * BM + row_in_tile;
        if (lrow < M_eff) {
            const int row = gp.tok_off + lrow;
            const int* idx = p.sorted_idx + static_cast<size_t>(row) * p.C;
            const float* beta = p.beta + static_cast<size_t>(row) * p.C;
            st.cursor = lower_bound_slot(idx, p.C, gp.b_off + n_blk * BN + gp.col_off);
            if (st.cursor < p.C) { st.next_col = __ldg(idx + st.cursor); st.beta_a = __ldg(beta + st.cursor); }
            if (st.cursor + 1 < p.C) { st.col_b = __ldg(idx + st.cursor + 1); st.beta_b = __ldg(beta + st.cursor + 1); }
            const float coef = p.coef[row];
            st.off = p.lse2[row] - log2f(fabsf(coef));              // coef == 0: +inf, the row's softmax part is +0
            st.sgn = coef < 0.f ? 0x80008000u : 0u;
        }
        return st;
    }
    // gp.row_off: ring buffer of this super-tile; gp.col_off, gp.N: first and number of the tile columns this warp handles
    static __device__ __forceinline__ void run(const Params& p, const GemmParams& gp, State st, uint32_t taddr,
                                               int m_blk, int n_blk, int row_in_tile, int, uint8_t*, int) {
        const int lrow = m_blk * BM + row_in_tile;
        const int row = gp.tok_off + lrow;
        const int* idx = p.sorted_idx + static_cast<size_t>(row) * p.C;          // dereferenced on live rows only (cursor < C)
        const float* beta = p.beta + static_cast<size_t>(row) * p.C;
        const float sgnf = st.sgn ? -1.f : 1.f;
        __nv_bfloat16* out = p.gs + static_cast<size_t>(gp.row_off) * p.planes * p.plane_stride + static_cast<size_t>(lrow) * p.ldg +
                             n_blk * BN + gp.col_off;
        for_each_chunk(taddr + gp.col_off, gp.N / 32, [&](float (&v)[32], int c) {
            const int col0 = gp.b_off + n_blk * BN + gp.col_off + c * 32;   // vocabulary column of v[0]
#pragma unroll
            for (int i = 0; i < 32; ++i) v[i] = ex2_approx(fmaf(v[i], LOG2E, -st.off));
            if (__any_sync(0xffffffffu, st.next_col < col0 + 32)) {
                while (st.next_col < col0 + 32) {                    // duplicates add up
                    add_at32(v, st.next_col - col0, sgnf * st.beta_a);
                    ++st.cursor;
                    st.next_col = st.col_b; st.beta_a = st.beta_b;    // the loads below are only waited for at a later hit
                    const bool more = st.cursor + 1 < p.C;
                    st.col_b = more ? __ldg(idx + st.cursor + 1) : IDX_SENTINEL;
                    st.beta_b = more ? __ldg(beta + st.cursor + 1) : 0.f;
                }
            }
            if (col0 + 32 > p.V) {
#pragma unroll
                for (int i = 0; i < 32; ++i)
                    if (col0 + i >= p.V) v[i] = 0.f;
            }
            if (lrow >= p.rows) return;                               // rows of a pair tile past the buffer are not stored
            if (p.planes == 1 && !p.st_hint) {                        // bf16 path: 64 bytes of this row, two 32-byte stores
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    uint32_t o[8];
#pragma unroll
                    for (int i = 0; i < 8; ++i) o[i] = pack_bf16x2(v[16 * q + 2 * i], v[16 * q + 2 * i + 1]) ^ st.sgn;
                    st_global_v8(out + c * 32 + 16 * q, o);
                }
                return;
            }
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
                // the sign of coef goes onto the packed pairs (the residuals above were taken in the sign-folded domain)
                uint4* dst = reinterpret_cast<uint4*>(out + pl * p.plane_stride + c * 32);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    if (p.st_hint) st_global_v4_hint(dst + q, w[4 * q] ^ st.sgn, w[4 * q + 1] ^ st.sgn, w[4 * q + 2] ^ st.sgn, w[4 * q + 3] ^ st.sgn, p.st_hint);
                    else dst[q] = make_uint4(w[4 * q] ^ st.sgn, w[4 * q + 1] ^ st.sgn, w[4 * q + 2] ^ st.sgn, w[4 * q + 3] ^ st.sgn);
                }
            }
#ifdef OPD_TRACE
        }, gp.tr);
#else
        });
#endif
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
        const int nchunks = min(BN / 32, (gp.N - n_blk * BN + 31) / 32);      // d % 64 == 0: chunks are all-in or all-out (warp-uniform)
#ifdef OPD_EXPERIMENTS
        if (p.dbg == 2) return;
        const bool reduce = !gp.first && p.dbg != 1;
#else
        const bool reduce = !gp.first;
#endif
        for_each_chunk(taddr, nchunks, [&](float (&v)[32], int c) {
            const int col0 = n_blk * BN + c * 32;
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
        });
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
        const int nchunks = min(BN / 32, (gp.N - n_blk * BN + 31) / 32);
#ifdef OPD_EXPERIMENTS
        if (p.dbg == 2) return;
        const bool reduce = !gp.first && p.dbg != 1;
#else
        const bool reduce = !gp.first;      // first token super-tile of an overwriting call: plain store
#endif
        for_each_chunk(taddr, nchunks, [&](float (&v)[32], int c) {
            if (warp_ok) stage_and_send(&p.m_gw, wbuf, c & 1, v, lane, gp.col_off + n_blk * BN + c * 32, gp.row_off + lrow0, reduce, p.hint);
        });
        drain_sends(lane);
    }
};

}  // namespace opd

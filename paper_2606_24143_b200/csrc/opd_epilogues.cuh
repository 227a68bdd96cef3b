// Tile epilogues of the OPD path.  Each runs on the 4 epilogue warps of a CTA: thread = one row of the CTA's
// 128 x 256 fp32 accumulator (half of a pair's 256 x 256 tile), read from TMEM in 8 chunks of 32 columns.
//   FwdEpi   z tile -> per-row (max, sum exp) partial of the tile + gather of the cached columns   (S2, S3)
//   GEpi     z tile -> G = (1/N)(alpha p + sum_j beta_j e_{a_j}) as bf16 into the L2-resident super-tile (S6)
//   DxEpi    grad_hidden super-tile accumulate / emit                                               (S7)
//   DwEpi    grad_W accumulate                                                                      (S8)
//   StoreEpi plain fp32 store (opd_debug_gemm)
#pragma once
#include <cuda_bf16.h>
#include "opd_gemm.cuh"

namespace opd {

constexpr float LOG2E = 1.4426950408889634f;
constexpr int IDX_SENTINEL = 0x7fffffff;

// v[i] for a run-time i without spilling v[] to local memory
__device__ __forceinline__ float select32(const float (&v)[32], int i) {
    float r = v[0];
#pragma unroll
    for (int j = 1; j < 32; ++j) r = (i == j) ? v[j] : r;
    return r;
}
__device__ __forceinline__ void add_at32(float (&v)[32], int i, float b) {
#pragma unroll
    for (int j = 0; j < 32; ++j) v[j] += (i == j) ? b : 0.f;
}
// first slot s in the ascending list idx[0..C) with idx[s] >= col  (C <= 64) = the number of entries below col.
// Counted over the whole row with independent (vector) loads: one memory latency per tile instead of the log2(C) + 1
// dependent ones of a binary search (at d <= 2048 the epilogue of a tile has less time than that took).
__device__ __forceinline__ int lower_bound_slot(const int* __restrict__ idx, int C, int col) {
    int n = 0;
    if ((C & 3) == 0) {
        const int4* q = reinterpret_cast<const int4*>(idx);       // rows of [T][C] int32 are 16-byte aligned when C % 4 == 0
#pragma unroll 4
        for (int j = 0; j < C / 4; ++j) {
            const int4 e = __ldg(q + j);
            n += (e.x < col) + (e.y < col) + (e.z < col) + (e.w < col);
        }
    } else {
#pragma unroll 4
        for (int j = 0; j < C; ++j) n += __ldg(idx + j) < col;
    }
    return n;
}

struct NoState {};

// ------------------------------------------------------------------------------------------ StoreEpi
struct StoreEpi {
    struct Params { float* out; long ldo; };
    using State = NoState;
    static __device__ __forceinline__ State prepare(const Params&, const GemmParams&, int, int, int, int) { return {}; }
    static __device__ __forceinline__ void run(const Params& p, const GemmParams& gp, const State&, uint32_t taddr,
                                               int m_blk, int n_blk, int row_in_tile, int M_eff, uint8_t*, int) {
        const int row = m_blk * BM + row_in_tile;
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
            float v[32];
            tmem_ld32(taddr + c * 32, v);
            tmem_ld_wait();
            const int col0 = n_blk * BN + c * 32;
            if (row < M_eff) {
#pragma unroll
                for (int i = 0; i < 32; ++i)
                    if (col0 + i < gp.N) p.out[row * p.ldo + col0 + i] = v[i];
            }
        }
    }
};

// ------------------------------------------------------------------------------------------ FwdEpi
// S2 (online log-sum-exp partial of this vocab tile) + S3 (gather of the cached columns out of the tile).
// The gathered value is the very fp32 accumulator the LSE partial sees.
struct FwdEpi {
    struct Params {
        float2* partials;        // [num_n][t_pad]  (max, sum exp(z - max)) per row and vocab tile
        int t_pad;
        const int* sorted_idx;   // [T][C] ascending per row, IDX_SENTINEL in unused slots
        float* zc;               // [T][C] gathered logits, in sorted-slot order
        int C;
        int V;
        float* dbg_logits;       // optional [T][V] dump (opd_debug_logits)
    };
    struct State { int cursor; int next_col; int col_b; };      // col_b: the cached column after next_col (prefetched)
    static __device__ __forceinline__ State prepare(const Params& p, const GemmParams& gp, int m_blk, int n_blk,
                                                    int row_in_tile, int M_eff) {
        State st{p.C, IDX_SENTINEL, IDX_SENTINEL};
        const int row = m_blk * BM + row_in_tile;
        if (row < M_eff) {
            const int* idx = p.sorted_idx + static_cast<size_t>(row) * p.C;
            st.cursor = lower_bound_slot(idx, p.C, n_blk * BN);
            st.next_col = st.cursor < p.C ? __ldg(idx + st.cursor) : IDX_SENTINEL;
            st.col_b = st.cursor + 1 < p.C ? __ldg(idx + st.cursor + 1) : IDX_SENTINEL;
        }
        return st;
    }
    static __device__ __forceinline__ void run(const Params& p, const GemmParams& gp, State st, uint32_t taddr,
                                               int m_blk, int n_blk, int row_in_tile, int M_eff, uint8_t*, int) {
        const int row = m_blk * BM + row_in_tile;
        const bool live = row < M_eff;
        const int* idx = p.sorted_idx + static_cast<size_t>(row) * p.C;
        float mx = -INFINITY, sum = 0.f;
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
            float v[32];
            tmem_ld32(taddr + c * 32, v);
            tmem_ld_wait();
            const int col0 = n_blk * BN + c * 32;
            if (col0 >= p.V) break;                                   // warp-uniform
            if (__any_sync(0xffffffffu, st.next_col < col0 + 32)) {
                while (st.next_col < col0 + 32) {                    // cached column inside this chunk
                    p.zc[static_cast<size_t>(row) * p.C + st.cursor] = select32(v, st.next_col - col0);
                    ++st.cursor;
                    st.next_col = st.col_b;                           // the load below is only waited for at a later hit
                    st.col_b = st.cursor + 1 < p.C ? __ldg(idx + st.cursor + 1) : IDX_SENTINEL;
                }
            }
            if (p.dbg_logits != nullptr && live) {
#pragma unroll
                for (int i = 0; i < 32; ++i)
                    if (col0 + i < p.V) p.dbg_logits[static_cast<size_t>(row) * p.V + col0 + i] = v[i];
            }
            if (col0 + 32 > p.V) {
#pragma unroll
                for (int i = 0; i < 32; ++i)
                    if (col0 + i >= p.V) v[i] = -INFINITY;
            }
            float cm = v[0];
#pragma unroll
            for (int i = 1; i < 32; ++i) cm = fmaxf(cm, v[i]);
            if (cm > mx) {
                sum *= exp2f((mx - cm) * LOG2E);
                mx = cm;
            }
            const float m2 = mx * LOG2E;
            float s0 = 0.f, s1 = 0.f;
#pragma unroll
            for (int i = 0; i < 32; i += 2) {
                s0 += exp2f(fmaf(v[i], LOG2E, -m2));
                s1 += exp2f(fmaf(v[i + 1], LOG2E, -m2));
            }
            sum += s0 + s1;
        }
        if (live) p.partials[static_cast<size_t>(n_blk) * p.t_pad + row] = make_float2(mx, sum);
    }
};

}  // namespace opd

// Cache producers: the steps either side of the learner path that build the finite caches it
// consumes, on the same streamed contraction (logits tiles in TMEM, never stored):
//   top-k cache   S = TopK(q(.|s), k) chosen by the scoring model + log q on S            (Fig. 1)
//   sample cache  a_1..a_K ~ p_old(.|s) iid WITH replacement + log p_old(a_j|s)
// Both run the forward contraction twice: pass A is gemm_kernel<FwdEpi> (per-tile (max, sum exp) partials -> lse),
// pass B re-streams the tiles with one of the epilogues below.
//   top-k:   theta_t = k-th largest TILE maximum of row t is a lower bound of the k-th largest logit (each of those k
//            tiles holds an element >= theta_t), so pass B only has to collect the few elements >= theta_t
//            (about k of them on smooth rows) into a bounded candidate list; k_topk_select ranks the candidates.
//   samples: inverse-CDF draws from caller-supplied uniforms u_tj: the tile masses of pass A locate the tile of each
//            draw (k_sample_targets), pass B resolves the column inside that tile by a prefix sum over its 256 logits.
#pragma once
#include "opd_estimators.cuh"

namespace opd {

// ------------------------------------------------------------------------------------------ lse of pass A
// lse_t from the per-tile partials; optionally theta_t = k-th largest tile maximum (k <= number of tiles, else -inf).
// One warp per row.
__global__ void __launch_bounds__(256) k_lse_theta(const float2* __restrict__ partials, int num_n, int t_pad, int T, int k,
                                                   float* __restrict__ lse, float* __restrict__ theta) {
    const int lane = threadIdx.x & 31;
    const int row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= T) return;
    float M = -INFINITY;
    for (int n = lane; n < num_n; n += 32) M = fmaxf(M, partials[static_cast<size_t>(n) * t_pad + row].x);
    for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
    float S = 0.f;
    for (int n = lane; n < num_n; n += 32) {
        const float2 q = partials[static_cast<size_t>(n) * t_pad + row];
        S += q.y * expf(q.x - M);
    }
    for (int o = 16; o > 0; o >>= 1) S += __shfl_xor_sync(0xffffffffu, S, o);
    if (lane == 0) lse[row] = M + logf(S);
    if (theta == nullptr) return;
    if (k > num_n) { if (lane == 0) theta[row] = -INFINITY; return; }
    // k selection passes over the tile maxima in the order (value descending, tile index ascending): pass i finds the
    // largest entry that comes after the one pass i-1 found; the k-th one is theta.
    float pv = INFINITY; int pi = -1;
    for (int it = 0; it < k; ++it) {
        float bv = -INFINITY; int bi = 0x7fffffff;
        for (int n = lane; n < num_n; n += 32) {
            const float m = partials[static_cast<size_t>(n) * t_pad + row].x;
            const bool after = (m < pv) || (m == pv && n > pi);
            if (after && (m > bv || (m == bv && n < bi))) { bv = m; bi = n; }
        }
        for (int o = 16; o > 0; o >>= 1) {
            const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
        }
        pv = bv; pi = bi;
    }
    if (lane == 0) theta[row] = pv;
}

// out[live_rows[i]] = in[i] for the live compact rows (lse_out in the caller's row order)
__global__ void __launch_bounds__(256) k_scatter_rows_f32(const float* __restrict__ in, const int* __restrict__ live_rows,
                                                          const int* __restrict__ n_live, int T, float* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < T && i < *n_live) out[live_rows[i]] = in[i];
}

// ------------------------------------------------------------------------------------------ CollectEpi (top-k pass B)
struct CollectEpi {
    struct Params {
        const float* theta;      // [T]
        int* count;              // [T] candidates appended so far (may exceed cap: overflow)
        float2* cand;            // [T][cap] (logit, column index as int bits)
        int cap;
        int V;
    };
    struct State { float theta; };
    static __device__ __forceinline__ State prepare(const Params& p, const GemmParams&, int m_blk, int, int row_in_tile, int M_eff) {
        const int row = m_blk * BM + row_in_tile;
        return State{row < M_eff ? p.theta[row] : INFINITY};
    }
    static __device__ __forceinline__ void run(const Params& p, const GemmParams&, State st, uint32_t taddr,
                                               int m_blk, int n_blk, int row_in_tile, int M_eff, uint8_t*, int) {
        const int row = m_blk * BM + row_in_tile;
        float2* cand = p.cand + static_cast<size_t>(row) * p.cap;
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
            float v[32];
            tmem_ld32(taddr + c * 32, v);
            tmem_ld_wait();
            const int col0 = n_blk * BN + c * 32;
            if (col0 >= p.V) break;                                   // warp-uniform
            float cm = -INFINITY;
#pragma unroll
            for (int i = 0; i < 32; ++i) {
                if (col0 + i >= p.V) v[i] = -INFINITY;
                cm = fmaxf(cm, v[i]);
            }
            if (row < M_eff && cm >= st.theta) {
#pragma unroll
                for (int i = 0; i < 32; ++i) {
                    if (v[i] >= st.theta && col0 + i < p.V) {          // rare: about k hits per row over the whole vocabulary
                        const int pos = atomicAdd(p.count + row, 1);
                        if (pos < p.cap) cand[pos] = make_float2(v[i], __int_as_float(col0 + i));
                    }
                }
            }
        }
    }
};

// Rank the candidates of each row: the k largest logits, ties -> lowest column first (the order a stable descending
// sort gives), written in descending order with their log-probs.  One warp per row.
__global__ void __launch_bounds__(256) k_topk_select(const float2* __restrict__ cand, const int* __restrict__ count, int cap, int T, int k,
                                                     const float* __restrict__ lse, const int* __restrict__ live_rows, const int* __restrict__ n_live,
                                                     int* __restrict__ idx_out, long ld_idx,
                                                     float* __restrict__ logp_out, long ld_logp, int* __restrict__ overflow) {
    const int lane = threadIdx.x & 31;
    const int row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);      // compact row
    if (row >= T || row >= *n_live) return;
    const int tok = live_rows[row];                                            // its row in the caller's arrays
    int n = count[row];
    if (n > cap) { if (lane == 0) atomicMax(overflow, n); n = cap; }
    const float2* c = cand + static_cast<size_t>(row) * cap;
    const float l = lse[row];
    for (int i = lane; i < n; i += 32) {
        const float vi = c[i].x;
        const int ci = __float_as_int(c[i].y);
        int rank = 0;
        for (int j = 0; j < n; ++j) {
            const float vj = c[j].x;
            rank += (vj > vi) || (vj == vi && __float_as_int(c[j].y) < ci);
        }
        if (rank < k) {
            idx_out[static_cast<size_t>(tok) * ld_idx + rank] = ci;
            logp_out[static_cast<size_t>(tok) * ld_logp + rank] = vi - l;
        }
    }
    for (int r = n + lane; r < k; r += 32) {      // fewer than k candidates (only if V < k)
        idx_out[static_cast<size_t>(tok) * ld_idx + r] = -1;
        logp_out[static_cast<size_t>(tok) * ld_logp + r] = -INFINITY;
    }
}

// ------------------------------------------------------------------------------------------ sampling: targets
// Per row: sort the K uniforms ascending (rank counting, keeps the permutation), then one sweep over the tile masses
// m_n = sumexp_n * exp(max_n - lse) assigns every draw its tile and the mass still to be covered inside that tile:
//   draw with target c = u * (sum_n m_n) lies in the first tile n with cum_n >= c;  residual = c - cum_{n-1}.
// One thread per row (K <= 64, num_n tiles).
__global__ void __launch_bounds__(128) k_sample_targets(const float2* __restrict__ partials, int num_n, int t_pad, int T, int K,
                                                        const float* __restrict__ lse, const int* __restrict__ live_rows,
                                                        const int* __restrict__ n_live, const float* __restrict__ u, long ld_u,
                                                        int* __restrict__ tgt_tile, float* __restrict__ tgt_res,
                                                        unsigned char* __restrict__ perm) {
    const int row = blockIdx.x * blockDim.x + threadIdx.x;                    // compact row
    if (row >= T || row >= *n_live) return;
    const float* ur = u + static_cast<size_t>(live_rows[row]) * ld_u;         // the uniforms are in the caller's row order
    int* tt = tgt_tile + static_cast<size_t>(row) * K;
    float* tr = tgt_res + static_cast<size_t>(row) * K;
    unsigned char* pr = perm + static_cast<size_t>(row) * K;
    for (int j = 0; j < K; ++j) {
        const float a = ur[j];
        int rank = 0;
        for (int q = 0; q < K; ++q) { const float b = ur[q]; rank += (b < a) || (b == a && q < j); }
        tr[rank] = a;                        // sorted uniforms for now
        pr[rank] = static_cast<unsigned char>(j);
    }
    const float l = lse[row];
    float total = 0.f;
    for (int n = 0; n < num_n; ++n) {
        const float2 q = partials[static_cast<size_t>(n) * t_pad + row];
        total += q.y * expf(q.x - l);
    }
    int s = 0;
    float cum = 0.f;
    for (int n = 0; n < num_n && s < K; ++n) {
        const float2 q = partials[static_cast<size_t>(n) * t_pad + row];
        const float before = cum;
        cum += q.y * expf(q.x - l);
        while (s < K && (tr[s] * total <= cum || n == num_n - 1)) {
            tt[s] = n;
            tr[s] = fmaxf(tr[s] * total - before, 0.f);
            ++s;
        }
    }
}

// ------------------------------------------------------------------------------------------ SampleEpi (sampling pass B)
// Resolves, inside the tile a draw fell into, the first column whose running mass reaches the residual.  The draws of a
// row are sorted, so one forward scan over the tile serves all of them; draws left over at the end of the tile
// (rounding between the two passes) take the tile's last valid column.
struct SampleEpi {
    struct Params {
        const int* tgt_tile;     // [T][K] ascending per row
        const float* tgt_res;    // [T][K]
        const unsigned char* perm;
        const float* lse;        // [T]
        int K;
        int V;
        int* idx_out; long ld_idx;
        float* logp_out; long ld_logp;
        const int* live_rows;    // compact row -> row of the caller's arrays
    };
    struct State { int cursor; float lse; int tok; };
    static __device__ __forceinline__ State prepare(const Params& p, const GemmParams&, int m_blk, int n_blk, int row_in_tile, int M_eff) {
        State st{p.K, 0.f, 0};
        const int row = m_blk * BM + row_in_tile;
        if (row < M_eff) {
            st.cursor = lower_bound_slot(p.tgt_tile + static_cast<size_t>(row) * p.K, p.K, n_blk);
            st.lse = p.lse[row];
            st.tok = p.live_rows[row];
        }
        return st;
    }
    static __device__ __forceinline__ void run(const Params& p, const GemmParams&, State st, uint32_t taddr,
                                               int m_blk, int n_blk, int row_in_tile, int M_eff, uint8_t*, int) {
        const int row = m_blk * BM + row_in_tile;
        const int* tt = p.tgt_tile + static_cast<size_t>(row) * p.K;
        const float* tr = p.tgt_res + static_cast<size_t>(row) * p.K;
        const unsigned char* pr = p.perm + static_cast<size_t>(row) * p.K;
        bool mine = row < M_eff && st.cursor < p.K && tt[st.cursor] == n_blk;      // a draw of this row lies in this tile
        if (!__any_sync(0xffffffffu, mine)) return;                                // nothing to resolve here
        float res = mine ? tr[st.cursor] : 0.f;
        float cum = 0.f;
        int last_col = -1; float last_z = 0.f;
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
            float v[32];
            tmem_ld32(taddr + c * 32, v);
            tmem_ld_wait();
            const int col0 = n_blk * BN + c * 32;
            if (col0 >= p.V) break;                                   // warp-uniform
            if (!mine) continue;
            const int nv = min(32, p.V - col0);                       // valid columns of this chunk
            float pre[32];                                            // running mass inside the chunk
            float run = 0.f;
#pragma unroll
            for (int i = 0; i < 32; ++i) {
                run += (i < nv) ? expf(v[i] - st.lse) : 0.f;
                pre[i] = run;
            }
            while (mine && cum + run >= res) {                        // this draw resolves inside the chunk
                int pos = 32;
#pragma unroll
                for (int i = 31; i >= 0; --i) pos = (cum + pre[i] >= res) ? i : pos;
                pos = min(pos, nv - 1);
                const float z = select32(v, pos);
                p.idx_out[static_cast<size_t>(st.tok) * p.ld_idx + pr[st.cursor]] = col0 + pos;
                p.logp_out[static_cast<size_t>(st.tok) * p.ld_logp + pr[st.cursor]] = z - st.lse;
                ++st.cursor;
                mine = st.cursor < p.K && tt[st.cursor] == n_blk;
                res = mine ? tr[st.cursor] : 0.f;
            }
            cum += run;
            last_col = col0 + nv - 1; last_z = select32(v, nv - 1);
        }
        while (mine) {                                                 // rounding: residual beyond the tile's mass
            p.idx_out[static_cast<size_t>(st.tok) * p.ld_idx + pr[st.cursor]] = last_col;
            p.logp_out[static_cast<size_t>(st.tok) * p.ld_logp + pr[st.cursor]] = last_z - st.lse;
            ++st.cursor;
            mine = st.cursor < p.K && tt[st.cursor] == n_blk;
        }
    }
};

}  // namespace opd

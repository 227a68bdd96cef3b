// Dense full-vocabulary forward KL from transmitted teacher hidden states (the direction the paper
// names as future work: "transmitting teacher hidden states and recomputing student logits"):
//     q_t = softmax(h^T_t . W_T)     p_t = softmax(x_t . W)      L_t = D_F = sum_v q_tv (log q_tv - log p_tv)   (Eq.(1))
//     dL_t/dz_tv = p_tv - q_tv
// Two heads are streamed; neither set of logits is ever stored.  The backward kernel gets a fourth tile type:
//     Q(s)   teacher logits of super-tile s -> q^ = round_bf16(exp(z^T - lse_T)) into a two-deep Q ring (consumed from L2),
//            and the row sums A_t += sum_v q^_tv (z^T_tv - lse_T)
//     G(s)   student logits recomputed -> G = (1/N)(exp(z - lse_p) - q^) into the G ring, B_t += sum_v q^_tv (z_tv - lse_p)
// followed by the unchanged grad_hidden / grad_W tiles.  L_t = A_t - B_t uses the SAME rounded q^ in both sums, so the
// bf16 rounding of q only perturbs the weights of the KL terms (relative 2^-9 per term), not the large entropy and
// cross-entropy sums separately.  With fp32 inputs the Q ring is fp32 and q^ = q.
//
// Reverse direction (OPD_F_DENSE_REVERSE; Eq.(2)):  L_t = D_R = sum_v p_tv (log p_tv - log q_tv),
//     dL_t/dz_tv = p_tv (log p_tv - log q_tv - L_t)       (the "+1" of Eq.(3) cancels against the softmax Jacobian)
// The Q tiles then store log q = z^T - lse_T (always fp32: a bf16 log-prob of magnitude ~10 would carry an absolute error of
// 0.03 into every term), a first launch of Q + G tiles accumulates L_t = sum_v p (log p - log q) without storing G, and the
// backward launch re-forms Q, then G = (1/N) p (log p - log q - L_t), followed by the unchanged grad_hidden / grad_W tiles.
#pragma once
#include "opd_epilogues_bwd.cuh"

namespace opd {

// per compact row: lse * log2(e) of both heads and 1/N
__global__ void __launch_bounds__(256) k_dense_rows(const float* __restrict__ lse_p, const float* __restrict__ lse_t, const int* __restrict__ n_live,
                                                    float norm_override, int t_pad, float* __restrict__ lse2_p, float* __restrict__ lse2_t,
                                                    float* __restrict__ coef, float* __restrict__ acc_a, float* __restrict__ acc_b) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= t_pad) return;
    const int n = *n_live;
    const float norm = norm_override > 0.f ? norm_override : static_cast<float>(n);
    const bool live = i < n;
    lse2_p[i] = live ? lse_p[i] * LOG2E : 0.f;
    lse2_t[i] = live ? lse_t[i] * LOG2E : 0.f;
    coef[i] = (live && norm > 0.f) ? 1.f / norm : 0.f;
    acc_a[i] = 0.f; acc_b[i] = 0.f;
}

// ------------------------------------------------------------------------------------------ QEpi
struct QEpi {
    struct Params {
        void* qs;                // Q ring buffer of this tile: [rows][ldq] bf16 (or fp32)
        int rows; long ldq; int q_fp32;
        const float* lse2_t;     // [T] teacher lse * log2(e), compact rows
        float* acc_a;            // [T] A_t (forward direction)
        int V;
        int logq;                // reverse direction: store log q (fp32 ring) instead of q, no A_t
    };
    struct State { float lse2; };
    static __device__ __forceinline__ State prepare(const Params& p, const GemmParams& gp, int m_blk, int, int row_in_tile, int M_eff) {
        const int lrow = m_blk * BM + row_in_tile;
        return State{lrow < M_eff ? p.lse2_t[gp.tok_off + lrow] : 0.f};
    }
    static __device__ __forceinline__ void run(const Params& p, const GemmParams& gp, State st, uint32_t taddr,
                                               int m_blk, int n_blk, int row_in_tile, int M_eff, uint8_t*, int) {
        const int lrow = m_blk * BM + row_in_tile;
        const bool live = lrow < M_eff;
        float a = 0.f;
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
            float v[32];
            tmem_ld32(taddr + c * 32, v);
            tmem_ld_wait();
            const int col0 = gp.b_off + n_blk * BN + c * 32;
            uint32_t w[16];
#pragma unroll
            for (int i = 0; i < 32; i += 2) {
                float q0 = 0.f, q1 = 0.f;
                if (p.logq) {                                     // log q_tv = z^T_tv - lse_T
                    if (live && col0 + i < p.V) q0 = v[i] - st.lse2 * (1.f / LOG2E);
                    if (live && col0 + i + 1 < p.V) q1 = v[i + 1] - st.lse2 * (1.f / LOG2E);
                    v[i] = q0; v[i + 1] = q1;
                    continue;
                }
                if (live && col0 + i < p.V) q0 = exp2f(fmaf(v[i], LOG2E, -st.lse2));
                if (live && col0 + i + 1 < p.V) q1 = exp2f(fmaf(v[i + 1], LOG2E, -st.lse2));
                if (!p.q_fp32) {                                  // the rounded value is the one every later use sees
                    w[i >> 1] = pack_bf16x2(q0, q1);
                    const __nv_bfloat162 t = *reinterpret_cast<const __nv_bfloat162*>(&w[i >> 1]);
                    q0 = __low2float(t); q1 = __high2float(t);
                }
                a = fmaf(q0, v[i] - st.lse2 * (1.f / LOG2E), a);
                a = fmaf(q1, v[i + 1] - st.lse2 * (1.f / LOG2E), a);
                v[i] = q0; v[i + 1] = q1;
            }
            if (lrow >= p.rows) continue;
            if (p.q_fp32) {
                float4* dst = reinterpret_cast<float4*>(static_cast<float*>(p.qs) + static_cast<size_t>(lrow) * p.ldq + n_blk * BN + c * 32);
#pragma unroll
                for (int q = 0; q < 8; ++q) dst[q] = make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
            } else {
                uint4* dst = reinterpret_cast<uint4*>(static_cast<__nv_bfloat16*>(p.qs) + static_cast<size_t>(lrow) * p.ldq + n_blk * BN + c * 32);
#pragma unroll
                for (int q = 0; q < 4; ++q) dst[q] = make_uint4(w[4 * q], w[4 * q + 1], w[4 * q + 2], w[4 * q + 3]);
            }
        }
        if (live && !p.logq) atomicAdd(p.acc_a + gp.tok_off + lrow, a);
    }
};

// ------------------------------------------------------------------------------------------ GDenseEpi
struct GDenseEpi {
    struct Params {
        __nv_bfloat16* gs;       // G ring buffer of this tile: [planes][rows][ldg]
        int rows; long ldg; long plane_stride; int planes;
        const void* qs;          // Q ring buffer of the same super-tile
        long ldq; int q_fp32;
        const float* lse2_p;     // [T] student lse * log2(e)
        const float* coef;       // [T] 1/N (0 on dead rows)
        float* acc_b;            // [T] B_t (forward) / L_t (reverse, first launch); null: not accumulated
        int V;
        int reverse;             // the Q ring holds log q; G = coef * p * (log p - log q - L_t)
        const float* lt;         // [T] L_t of the reverse direction (second launch), compact rows
    };
    struct State { float lse2; float coef; float lt; };
    static __device__ __forceinline__ State prepare(const Params& p, const GemmParams& gp, int m_blk, int, int row_in_tile, int M_eff) {
        const int lrow = m_blk * BM + row_in_tile;
        State st{0.f, 0.f, 0.f};
        if (lrow < M_eff) {
            st.lse2 = p.lse2_p[gp.tok_off + lrow]; st.coef = p.coef[gp.tok_off + lrow];
            if (p.reverse && p.lt) st.lt = p.lt[gp.tok_off + lrow];
        }
        return st;
    }
    static __device__ __forceinline__ void run(const Params& p, const GemmParams& gp, State st, uint32_t taddr,
                                               int m_blk, int n_blk, int row_in_tile, int M_eff, uint8_t*, int) {
        const int lrow = m_blk * BM + row_in_tile;
        const bool live = lrow < M_eff;
        const bool stored = lrow < p.rows;
        __nv_bfloat16* out = p.gs + static_cast<size_t>(lrow) * p.ldg + n_blk * BN;
        float b = 0.f;
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
            float v[32];
            tmem_ld32(taddr + c * 32, v);
            tmem_ld_wait();
            const int col0 = gp.b_off + n_blk * BN + c * 32;
            float q[32];
            if (live) {                                            // rows past the live count were stored as zeros by QEpi
                if (p.q_fp32) {
                    const float4* src = reinterpret_cast<const float4*>(static_cast<const float*>(p.qs) + static_cast<size_t>(lrow) * p.ldq + n_blk * BN + c * 32);
#pragma unroll
                    for (int j = 0; j < 8; ++j) { const float4 t = __ldcg(src + j); q[4 * j] = t.x; q[4 * j + 1] = t.y; q[4 * j + 2] = t.z; q[4 * j + 3] = t.w; }
                } else {
                    const uint4* src = reinterpret_cast<const uint4*>(static_cast<const __nv_bfloat16*>(p.qs) + static_cast<size_t>(lrow) * p.ldq + n_blk * BN + c * 32);
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const uint4 t = __ldcg(src + j);            // written through L2 by other SMs: bypass L1
                        const uint32_t ww[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const __nv_bfloat162 h2 = *reinterpret_cast<const __nv_bfloat162*>(&ww[e]);
                            q[8 * j + 2 * e] = __low2float(h2); q[8 * j + 2 * e + 1] = __high2float(h2);
                        }
                    }
                }
            }
#pragma unroll
            for (int i = 0; i < 32; ++i) {
                if (live && col0 + i < p.V) {
                    if (p.reverse) {
                        const float pr = exp2f(fmaf(v[i], LOG2E, -st.lse2));
                        const float tdiff = (v[i] - st.lse2 * (1.f / LOG2E)) - q[i];      // log p - log q
                        b = fmaf(pr, tdiff, b);
                        v[i] = st.coef * pr * (tdiff - st.lt);
                    } else {
                        b = fmaf(q[i], v[i] - st.lse2 * (1.f / LOG2E), b);
                        v[i] = st.coef * (exp2f(fmaf(v[i], LOG2E, -st.lse2)) - q[i]);
                    }
                } else {
                    v[i] = 0.f;
                }
            }
            if (!stored) continue;
            for (int pl = 0; pl < p.planes; ++pl) {
                uint32_t w[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    w[i] = pack_bf16x2(v[2 * i], v[2 * i + 1]);
                    if (pl + 1 < p.planes) {
                        __nv_bfloat162 t = *reinterpret_cast<__nv_bfloat162*>(&w[i]);
                        v[2 * i] -= __low2float(t);
                        v[2 * i + 1] -= __high2float(t);
                    }
                }
                uint4* dst = reinterpret_cast<uint4*>(out + pl * p.plane_stride + c * 32);
#pragma unroll
                for (int qq = 0; qq < 4; ++qq) dst[qq] = make_uint4(w[4 * qq], w[4 * qq + 1], w[4 * qq + 2], w[4 * qq + 3]);
            }
        }
        if (live && p.acc_b) atomicAdd(p.acc_b + gp.tok_off + lrow, b);
    }
};

// L_t = A_t - B_t (forward; reverse: L_t = B_t) in caller order, block sums for the deterministic loss reduction
// (k_loss_final finishes it); lt (optional, compact rows) keeps L_t for the reverse direction's gradient tiles
__global__ void __launch_bounds__(128) k_dense_loss(const float* __restrict__ acc_a, const float* __restrict__ acc_b, int reverse,
                                                    const int* __restrict__ live_rows, const int* __restrict__ n_live,
                                                    float* __restrict__ per_token_kl, float* __restrict__ lt, double* __restrict__ block_sums) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    float L = 0.f;
    if (i < *n_live) {
        L = reverse ? acc_b[i] : acc_a[i] - acc_b[i];
        per_token_kl[live_rows[i]] = L;
    }
    if (lt != nullptr && i < gridDim.x * blockDim.x) lt[i] = L;
    __shared__ double sh[128];
    sh[threadIdx.x] = static_cast<double>(L);
    __syncthreads();
    for (int s = 64; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) block_sums[blockIdx.x] = sh[0];
}

}  // namespace opd

// Non-GEMM kernels of the OPD path: S0 pre-pass (live-row compaction, cache sort, operand staging),
// S4 estimators + S5 loss reduction.  All O(T*C) or O(T*d) streaming work.
#pragma once
#include <cuda_bf16.h>
#include <cstdint>
#include "opd_epilogues.cuh"

namespace opd {

// flags / modes restated from include/opd.h (kept numerically identical there)
constexpr int MODE_FKL = 0, MODE_MC = 1, MODE_MIXED = 2, MODE_RKL_TOPK = 3;
constexpr unsigned FL_NO_RENORM_TEACHER = 1, FL_RENORM_STUDENT = 2, FL_SUR_CLIP = 64, FL_SUR_A_OLD = 128;
constexpr float CLIP_EPS = 0.2f;

// ------------------------------------------------------------------------------------------ S0a
// Ordered compaction of live rows: live_rows[i] = i-th token with mask != 0; *n_live = count.  One block.
__global__ void __launch_bounds__(1024) k_compact(const unsigned char* __restrict__ mask, int T, int all_live,
                                                  int* __restrict__ live_rows, int* __restrict__ n_live) {
    __shared__ int warp_cnt[32];
    __shared__ int base;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) base = 0;
    __syncthreads();
    for (int t0 = 0; t0 < T; t0 += 1024) {
        const int t = t0 + threadIdx.x;
        const bool live = t < T && (all_live || mask[t] != 0);
        const unsigned b = __ballot_sync(0xffffffffu, live);
        if (lane == 0) warp_cnt[warp] = __popc(b);
        __syncthreads();
        int off = base;
        for (int w = 0; w < warp; ++w) off += warp_cnt[w];
        if (live) live_rows[off + __popc(b & ((1u << lane) - 1))] = t;
        __syncthreads();
        if (threadIdx.x == 0) {
            int s = 0;
            for (int w = 0; w < 32; ++w) s += warp_cnt[w];
            base += s;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) *n_live = base;
}

// three-term bf16 split of an fp32 value: x = b0 + b1 + b2 (exact up to underflow)
__device__ __forceinline__ void split3(float x, __nv_bfloat16& b0, __nv_bfloat16& b1, __nv_bfloat16& b2) {
    b0 = __float2bfloat16_rn(x);
    const float r1 = x - __bfloat162float(b0);
    b1 = __float2bfloat16_rn(r1);
    b2 = __float2bfloat16_rn(r1 - __bfloat162float(b1));
}

// ------------------------------------------------------------------------------------------ S0b
// Compacted copy of hidden: xc[plane][i][:] = hidden[live_rows[i]][:] for i < n_live, zeros for n_live <= i < t_pad.
// fp32 input is split into 3 bf16 planes.  One block per compact row.
__global__ void __launch_bounds__(256) k_gather_rows(const void* __restrict__ hidden, long ld_hidden, int is_fp32, int d,
                                                     int t_pad, const int* __restrict__ live_rows, const int* __restrict__ n_live,
                                                     __nv_bfloat16* __restrict__ xc, long plane_stride) {
    const int i = blockIdx.x;
    const bool live = i < *n_live;
    const int tok = live ? live_rows[i] : 0;
    __nv_bfloat16* dst = xc + static_cast<size_t>(i) * d;
    if (!is_fp32) {
        const uint4* src = reinterpret_cast<const uint4*>(static_cast<const __nv_bfloat16*>(hidden) + static_cast<size_t>(tok) * ld_hidden);
        uint4* d4 = reinterpret_cast<uint4*>(dst);
        for (int k = threadIdx.x; k < d / 8; k += blockDim.x) d4[k] = live ? src[k] : make_uint4(0, 0, 0, 0);
    } else {
        const float* src = static_cast<const float*>(hidden) + static_cast<size_t>(tok) * ld_hidden;
        for (int k = threadIdx.x; k < d; k += blockDim.x) {
            __nv_bfloat16 b0, b1, b2;
            split3(live ? src[k] : 0.f, b0, b1, b2);
            dst[k] = b0; dst[plane_stride + k] = b1; dst[2 * plane_stride + k] = b2;
        }
    }
}

// fp32 W (any of the two layouts, `rows` x `cols` with row stride ld) -> 3 contiguous bf16 planes [rows][cols]
__global__ void __launch_bounds__(256) k_split_matrix(const float* __restrict__ src, long ld, int rows, int cols,
                                                      __nv_bfloat16* __restrict__ dst, long plane_stride) {
    const size_t n = static_cast<size_t>(rows) * cols;
    for (size_t e = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; e < n; e += static_cast<size_t>(gridDim.x) * blockDim.x) {
        const size_t r = e / cols, c = e - r * cols;
        __nv_bfloat16 b0, b1, b2;
        split3(src[r * ld + c], b0, b1, b2);
        dst[e] = b0; dst[plane_stride + e] = b1; dst[2 * plane_stride + e] = b2;
    }
}

// Zero an fp32 matrix (rows x cols, row stride ld).  With `only_if_empty` set, only when *only_if_empty == 0: the dense
// backward overwrites grad_W itself (its first token super-tile stores) unless the call has no live token at all.
__global__ void __launch_bounds__(256) k_zero_matrix(float* __restrict__ m, long ld, int rows, int cols, const int* __restrict__ only_if_empty) {
    if (only_if_empty != nullptr && *only_if_empty != 0) return;
    const size_t n4 = static_cast<size_t>(rows) * (cols / 4);
    for (size_t e = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; e < n4; e += static_cast<size_t>(gridDim.x) * blockDim.x) {
        const size_t r = e / (cols / 4), c = e - r * (cols / 4);
        reinterpret_cast<float4*>(m + r * ld)[c] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

// out (bf16, row stride ldo) = round(acc) or round(out + acc): the final emit of OPD_F_GRADW_BF16 (sums are kept in fp32)
__global__ void __launch_bounds__(256) k_emit_bf16(const float* __restrict__ acc, long lda, int rows, int cols,
                                                   __nv_bfloat16* __restrict__ out, long ldo, int accumulate) {
    const size_t n8 = static_cast<size_t>(rows) * (cols / 8);
    for (size_t e = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; e < n8; e += static_cast<size_t>(gridDim.x) * blockDim.x) {
        const size_t r = e / (cols / 8), c = (e - r * (cols / 8)) * 8;
        const float4 a0 = *reinterpret_cast<const float4*>(acc + r * lda + c), a1 = *reinterpret_cast<const float4*>(acc + r * lda + c + 4);
        float v[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
        uint4* o = reinterpret_cast<uint4*>(out + r * ldo + c);
        if (accumulate) {
            const uint4 old = *o;
            const uint32_t w[4] = {old.x, old.y, old.z, old.w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const __nv_bfloat162 h2 = *reinterpret_cast<const __nv_bfloat162*>(&w[i]);
                v[2 * i] += __low2float(h2); v[2 * i + 1] += __high2float(h2);
            }
        }
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) { __nv_bfloat162 t = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]); w[i] = *reinterpret_cast<uint32_t*>(&t); }
        *o = make_uint4(w[0], w[1], w[2], w[3]);
    }
}

// ------------------------------------------------------------------------------------------ S0c
// Per live row: ascending (stable) sort of the first C_row cache indices by rank counting; keeps the
// permutation so outputs go back in caller slot order.  One warp per compact row.
__global__ void __launch_bounds__(256) k_sort_cache(const int* __restrict__ cache_idx, long ld_cache, const unsigned char* __restrict__ mask,
                                                    int mode, int k_fkl, int K_mc, int C, int V,
                                                    const int* __restrict__ live_rows, const int* __restrict__ n_live,
                                                    int* __restrict__ sorted_idx, unsigned char* __restrict__ perm,
                                                    int* __restrict__ bad_index_flag) {
    const int lane = threadIdx.x & 31;
    const int i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (i >= *n_live) return;
    const int tok = live_rows[i];
    int Crow = C;
    if (mode == MODE_MIXED) Crow = (mask[tok] == 1) ? k_fkl : K_mc;
    const int* src = cache_idx + static_cast<size_t>(tok) * ld_cache;
    int* so = sorted_idx + static_cast<size_t>(i) * C;
    unsigned char* po = perm + static_cast<size_t>(i) * C;
    for (int j = lane; j < C; j += 32) {
        if (j >= Crow) { so[j] = IDX_SENTINEL; po[j] = static_cast<unsigned char>(j); }
    }
    for (int j = lane; j < Crow; j += 32) {
        int a = src[j];
        if (a < 0 || a >= V) { atomicOr(bad_index_flag, 1); a = IDX_SENTINEL - 1; }   // never gathered
        int rank = 0;
        for (int q = 0; q < Crow; ++q) {
            int b = src[q];
            if (b < 0 || b >= V) b = IDX_SENTINEL - 1;
            rank += (b < a) || (b == a && q < j);
        }
        so[rank] = a;
        po[rank] = static_cast<unsigned char>(j);
    }
}

}  // namespace opd

// S7/S8 when alpha_t == 0 for every row (OPD_RKL_TOPK; OPD_FKL_TOPK with OPD_F_RENORM_STUDENT): the full-vocabulary lse
// cancels, dL/dz has support on the cached columns only, and the dense re-formation of softmax tiles is skipped:
//   grad_hidden[t,:] = sum_j beta_tj W(:, a_tj)              a gather-sum per token            (k_sparse_gh)
//   grad_W(:, v)     = sum_{(t,j): a_tj = v} beta_tj x_t     a segmented sum per column        (k_sparse_gw)
// The (column, entry) pairs are sorted by column with a stable LSD radix sort (k_radix_*), so every column's terms are
// added in (token, slot) order by ONE block: no atomics, bit-reproducible, and grad_W is written exactly once (zeros
// where no token cached the column).  W is read as contiguous d-vectors per column: the caller's array when it is stored
// [V,d], else a transposed scratch copy (k_transpose); grad_W is written in the caller's layout directly.
// Hot columns (real top-k supports: a few tokens such as punctuation sit in the support of most rows, so one column's
// run holds 1e4-1e5 entries): the sorted entry array is cut into fixed segments of GW_SEG entries; every segment that
// lies inside ONE column's run is summed by its own block beforehand (k_sparse_gw_seg, the whole grid in parallel), and
// the column's block adds these partial sums in segment order instead of walking the entries.  Which segments qualify
// depends on the sorted keys only, so the summation order stays fixed and the result bit-reproducible; a support
// without such runs takes exactly the arithmetic path it took before.
#pragma once
#include "opd_small_kernels.cuh"

namespace opd {

template <typename T>
__device__ __forceinline__ float ld_as_float(const void* base, size_t i) {
    if constexpr (sizeof(T) == 2) return __bfloat162float(static_cast<const __nv_bfloat16*>(base)[i]);
    else return static_cast<const float*>(base)[i];
}

// four consecutive elements starting at element i (i % 4 == 0, base 16-byte aligned) as floats, one vector load
template <typename T>
__device__ __forceinline__ void ld4_as_float(const void* base, size_t i, float (&x)[4]) {
    if constexpr (sizeof(T) == 2) {
        const uint2 v = *reinterpret_cast<const uint2*>(static_cast<const __nv_bfloat16*>(base) + i);
        x[0] = __uint_as_float(v.x << 16); x[1] = __uint_as_float(v.x & 0xffff0000u);
        x[2] = __uint_as_float(v.y << 16); x[3] = __uint_as_float(v.y & 0xffff0000u);
    } else {
        const float4 v = *reinterpret_cast<const float4*>(static_cast<const float*>(base) + i);
        x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w;
    }
}

// grad_hidden row of one live token (one block per compact row); columns in ascending order: a fixed summation order
template <typename T>
__global__ void __launch_bounds__(256) k_sparse_gh(const void* __restrict__ Wt, long ldwt, int d, int C, const int* __restrict__ sorted_idx,
                                                   const float* __restrict__ beta, const int* __restrict__ live_rows,
                                                   const int* __restrict__ n_live, void* __restrict__ grad_hidden, long ld_gh) {
    const int i = blockIdx.x;
    if (i >= *n_live) return;
    const int tok = live_rows[i];
    const int* idx = sorted_idx + static_cast<size_t>(i) * C;
    const float* b = beta + static_cast<size_t>(i) * C;
    for (int k = threadIdx.x; k < d; k += blockDim.x) {
        float g = 0.f;
        for (int s = 0; s < C; ++s) {
            const int col = idx[s];
            if (col >= IDX_SENTINEL - 1) break;             // unused slots (and invalid indices) sort to the end
            g = fmaf(b[s], ld_as_float<T>(Wt, static_cast<size_t>(col) * ldwt + k), g);
        }
        if constexpr (sizeof(T) == 2) static_cast<__nv_bfloat16*>(grad_hidden)[static_cast<size_t>(tok) * ld_gh + k] = __float2bfloat16_rn(g);
        else static_cast<float*>(grad_hidden)[static_cast<size_t>(tok) * ld_gh + k] = g;
    }
}

// ------------------------------------------------------------------------------------------ sort keys
// key = cached column of entry e = (compact row, sorted slot), V for unused slots, invalid indices and rows past the live count
__global__ void __launch_bounds__(256) k_sparse_keys(const int* __restrict__ sorted_idx, int C, size_t N, const int* __restrict__ n_live, int V,
                                                     uint32_t* __restrict__ keys, uint32_t* __restrict__ vals) {
    const size_t e = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x;
    if (e >= N) return;
    int col = V;
    if (static_cast<int>(e / C) < *n_live) {
        col = sorted_idx[e];
        if (col < 0 || col >= V) col = V;
    }
    keys[e] = static_cast<uint32_t>(col);
    vals[e] = static_cast<uint32_t>(e);
}

// ------------------------------------------------------------------------------------------ stable LSD radix sort, 8 bits per pass
constexpr int RS_TILE = 2048;      // elements per block: 8 warps x 8 chunks of 32

__global__ void __launch_bounds__(256) k_radix_hist(const uint32_t* __restrict__ keys, size_t N, int shift, uint32_t* __restrict__ hist, int nblk) {
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const size_t base = static_cast<size_t>(blockIdx.x) * RS_TILE;
    for (int j = 0; j < RS_TILE / 256; ++j) {
        const size_t e = base + j * 256 + threadIdx.x;
        if (e < N) atomicAdd(&h[(keys[e] >> shift) & 255u], 1u);        // integer counts: order-independent
    }
    __syncthreads();
    hist[static_cast<size_t>(threadIdx.x) * nblk + blockIdx.x] = h[threadIdx.x];     // digit-major: a scan gives stable offsets
}

// exclusive scan of n counters in place (one block; n = 256 * #blocks of the sort)
__global__ void __launch_bounds__(1024) k_radix_scan(uint32_t* __restrict__ a, size_t n) {
    __shared__ uint32_t sh[1024];
    __shared__ uint32_t carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (size_t b = 0; b < n; b += 1024) {
        const size_t i = b + threadIdx.x;
        const uint32_t v = i < n ? a[i] : 0u;
        sh[threadIdx.x] = v;
        __syncthreads();
        for (int off = 1; off < 1024; off <<= 1) {
            const uint32_t t = threadIdx.x >= off ? sh[threadIdx.x - off] : 0u;
            __syncthreads();
            sh[threadIdx.x] += t;
            __syncthreads();
        }
        if (i < n) a[i] = carry + sh[threadIdx.x] - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry += sh[1023];
        __syncthreads();
    }
}

__global__ void __launch_bounds__(256) k_radix_scatter(const uint32_t* __restrict__ keys, const uint32_t* __restrict__ vals, size_t N, int shift,
                                                       const uint32_t* __restrict__ hist, int nblk,
                                                       uint32_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out) {
    __shared__ uint32_t wh[8][256];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int j = threadIdx.x; j < 8 * 256; j += 256) (&wh[0][0])[j] = 0;
    __syncthreads();
    const size_t wbase = static_cast<size_t>(blockIdx.x) * RS_TILE + static_cast<size_t>(warp) * 256;
    // per-warp digit counts of its 256 consecutive elements
    for (int c = 0; c < 8; ++c) {
        const size_t e = wbase + c * 32 + lane;
        const uint32_t dg = e < N ? ((keys[e] >> shift) & 255u) : 256u;
        const uint32_t peers = __match_any_sync(0xffffffffu, dg);
        if (dg < 256u && lane == __ffs(peers) - 1) wh[warp][dg] += __popc(peers);
        __syncwarp();
    }
    __syncthreads();
    {   // first output position of (this block, warp w, digit): global offset of the block's digit + the earlier warps' counts
        uint32_t base = hist[static_cast<size_t>(threadIdx.x) * nblk + blockIdx.x];
        for (int w = 0; w < 8; ++w) { const uint32_t t = wh[w][threadIdx.x]; wh[w][threadIdx.x] = base; base += t; }
    }
    __syncthreads();
    for (int c = 0; c < 8; ++c) {
        const size_t e = wbase + c * 32 + lane;
        const bool valid = e < N;
        const uint32_t key = valid ? keys[e] : 0u;
        const uint32_t dg = valid ? ((key >> shift) & 255u) : 256u;
        const uint32_t peers = __match_any_sync(0xffffffffu, dg);
        uint32_t pos = 0;
        if (valid) pos = wh[warp][dg] + __popc(peers & ((1u << lane) - 1u));      // lanes in order: stable
        __syncwarp();
        if (valid && lane == __ffs(peers) - 1) wh[warp][dg] += __popc(peers);
        __syncwarp();
        if (valid) { keys_out[pos] = key; vals_out[pos] = vals[e]; }
    }
}

// ------------------------------------------------------------------------------------------ grad_W, column by column
// One block per group of 8 consecutive vocabulary columns: its sorted entries are a contiguous run; the terms of a column
// are added in run order (token, slot).  [d,V] storage: the 8 columns of a k-chunk are staged in shared memory and
// written as 32-byte rows; [V,d] storage: each column's d-vector is written directly.
constexpr int GW_KCHUNK = 1024;    // k values per pass of a block (4 per thread)
constexpr int GW_SEG = 256;        // entries per segment of the sorted entry array (hot columns: summed per segment first)

// Partial sums of the segments that lie inside one column's run: part[s][0..d) = sum over the GW_SEG entries of segment s, in
// entry order, of beta * x.  Grid (N / GW_SEG, ceil(d / GW_KCHUNK)); blocks of other segments return at once.
template <typename T>
__global__ void __launch_bounds__(256) k_sparse_gw_seg(const uint32_t* __restrict__ scol, const uint32_t* __restrict__ sent, int V, int C,
                                                       const float* __restrict__ beta, const int* __restrict__ live_rows,
                                                       const void* __restrict__ hidden, long ld_hidden, int d, float* __restrict__ part) {
    __shared__ float sb[GW_SEG];
    __shared__ size_t srow[GW_SEG];
    const size_t e0 = static_cast<size_t>(blockIdx.x) * GW_SEG;
    const uint32_t col = scol[e0];
    if (col >= static_cast<uint32_t>(V) || scol[e0 + GW_SEG - 1] != col) return;      // sorted: first == last means one column
    for (int i = threadIdx.x; i < GW_SEG; i += 256) {
        const uint32_t ent = sent[e0 + i];
        sb[i] = beta[ent];
        srow[i] = static_cast<size_t>(live_rows[ent / C]) * ld_hidden;
    }
    __syncthreads();
    const int k = blockIdx.y * GW_KCHUNK + threadIdx.x * 4;
    if (k >= d) return;
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll 4
    for (int i = 0; i < GW_SEG; ++i) {
        float x[4];
        ld4_as_float<T>(hidden, srow[i] + k, x);
        const float b = sb[i];
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[j] = fmaf(b, x[j], acc[j]);
    }
    *reinterpret_cast<float4*>(part + static_cast<size_t>(blockIdx.x) * d + k) = make_float4(acc[0], acc[1], acc[2], acc[3]);
}

template <typename T>
__global__ void __launch_bounds__(256) k_sparse_gw(const uint32_t* __restrict__ scol, const uint32_t* __restrict__ sent, size_t N, int V, int C,
                                                   const float* __restrict__ beta, const int* __restrict__ live_rows,
                                                   const void* __restrict__ hidden, long ld_hidden, int d,
                                                   const float* __restrict__ part, float* __restrict__ gw, long ldgw, int wl, int accumulate) {
    __shared__ size_t range[2];
    __shared__ float tile[GW_KCHUNK][8 + 1];
    const uint32_t c0 = blockIdx.x * 8u;
    if (threadIdx.x < 2) {                                  // lower_bound of c0 and c0 + 8 in the sorted columns
        const uint32_t target = c0 + 8u * threadIdx.x;
        size_t lo = 0, hi = N;
        while (lo < hi) { const size_t mid = (lo + hi) >> 1; if (scol[mid] < target) lo = mid + 1; else hi = mid; }
        range[threadIdx.x] = lo;
    }
    __syncthreads();
    const size_t lo = range[0], hi = range[1];
    for (int k0 = 0; k0 < d; k0 += GW_KCHUNK) {
        const int k = k0 + threadIdx.x * 4;
        const bool kin = k < d;                             // d % 64 == 0: a thread's 4 values are all in or all out
        float acc[4] = {0.f, 0.f, 0.f, 0.f};
        uint32_t cur = c0;
        auto flush = [&](uint32_t col) {                    // column `col` of this group is complete for this thread's k values
            if (wl == 0) {
#pragma unroll
                for (int j = 0; j < 4; ++j) tile[threadIdx.x * 4 + j][col - c0] = acc[j];
            } else if (kin) {
                float4* o = reinterpret_cast<float4*>(gw + static_cast<size_t>(col) * ldgw + k);
                float4 v = make_float4(acc[0], acc[1], acc[2], acc[3]);
                if (accumulate) { const float4 old = *o; v.x += old.x; v.y += old.y; v.z += old.z; v.w += old.w; }
                *o = v;
            }
            acc[0] = acc[1] = acc[2] = acc[3] = 0.f;
        };
        for (size_t e = lo; e < hi;) {
            const uint32_t col = scol[e];
            while (cur < col) { flush(cur); ++cur; }
            if (e % GW_SEG == 0 && e + GW_SEG <= hi && scol[e + GW_SEG - 1] == col) {
                // a whole segment of this column: k_sparse_gw_seg has summed it (same test there, on the sorted keys only)
                if (kin) {
                    const float4 p = *reinterpret_cast<const float4*>(part + (e / GW_SEG) * d + k);
                    acc[0] += p.x; acc[1] += p.y; acc[2] += p.z; acc[3] += p.w;
                }
                e += GW_SEG;
                continue;
            }
            if (kin) {
                const uint32_t ent = sent[e];
                const float b = beta[ent];
                float x[4];
                ld4_as_float<T>(hidden, static_cast<size_t>(live_rows[ent / C]) * ld_hidden + k, x);
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[j] = fmaf(b, x[j], acc[j]);
            }
            ++e;
        }
        while (cur < c0 + 8u) { flush(cur); ++cur; }
        if (wl == 0) {                                      // rows of 8 floats: grad_W[k][c0 .. c0 + 8)
            __syncthreads();
            for (int r = threadIdx.x; r < GW_KCHUNK && k0 + r < d; r += 256) {
                float* o = gw + static_cast<size_t>(k0 + r) * ldgw + c0;
#pragma unroll
                for (int j = 0; j < 8; ++j) o[j] = accumulate ? o[j] + tile[r][j] : tile[r][j];
            }
            __syncthreads();
        }
    }
}

// dst[c][r] = src[r][c] for an R x Cn matrix (row strides lds / ldd), 32 x 32 tiles through shared memory.
// Launch: grid (ceil(Cn/32), ceil(R/32)), block (32, 8).
template <typename T>
__global__ void __launch_bounds__(256) k_transpose(const T* __restrict__ src, long lds, int R, int Cn, T* __restrict__ dst, long ldd) {
    __shared__ T tile[32][33];
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    for (int y = threadIdx.y; y < 32; y += 8) {
        const int r = r0 + y, c = c0 + threadIdx.x;
        if (r < R && c < Cn) tile[y][threadIdx.x] = src[static_cast<size_t>(r) * lds + c];
    }
    __syncthreads();
    for (int y = threadIdx.y; y < 32; y += 8) {
        const int c = c0 + y, r = r0 + threadIdx.x;
        if (r < R && c < Cn) dst[static_cast<size_t>(c) * ldd + r] = tile[threadIdx.x][y];
    }
}

}  // namespace opd

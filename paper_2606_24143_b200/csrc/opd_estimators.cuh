// S2 (combine of the per-tile LSE partials), S4 (estimators per token), S5 (loss reduction).
//   FKL_TOPK  PAPER.md:57 Eq.(1) on the cached support, renormalisers Eq.(9)
//   RKL_MC    PAPER.md:191, Eq.(15); A_theta recomputed at learner time, rho unclipped
//             (PAPER.md:126-130); optional PPO clip / A_old variants of Eq.(6),(7) PAPER.md:132-141
//   RKL_TOPK  sparse top-k reverse KL on the cached support, App. A.1 Eq.(8)-(10) PAPER.md:289-303
// Output of S4 for the backward: dL_t/dz_v = alpha_t p_v + sum_j beta_tj [a_tj = v]  (both scaled by 1/N).
#pragma once
#include "opd_small_kernels.cuh"

namespace opd {

struct EstParams {
    const float2* partials; int num_n; int t_pad;       // [num_n][t_pad]
    const float* zc;                                     // [T][C] gathered logits, sorted-slot order
    const unsigned char* perm;                           // [T][C] sorted slot -> caller slot
    const float* lam; const float* old; long ld_cache;   // caller arrays [T][ld_cache]
    const unsigned char* mask;
    const int* live_rows; const int* n_live;
    int mode, k_fkl, K_mc, C;
    unsigned flags;
    float norm_override;
    // outputs
    float* lse2; float* coef; float* beta;               // compact-row order ([T], [T], [T][C])
    float* per_token_kl; float* lse_out; float* slp_out; // caller order; lse_out / slp_out may be null
    float* rho_out; long ld_rho; float* var1_out;        // optional diagnostics (opd_set_diagnostics), caller order
    float* seq_l1; float* seq_var1;                      // optional [T] (opd_set_seq_diagnostics): first-draw estimate, Eq.(16) variance
    double* block_sums;                                  // [gridDim.x]
};

__global__ void __launch_bounds__(128) k_estimator(const EstParams p) {
    const int n_live = *p.n_live;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const float norm = p.norm_override > 0.f ? p.norm_override : static_cast<float>(n_live);
    const float rs = norm > 0.f ? 1.f / norm : 0.f;
    float L = 0.f;
    if (i < n_live) {
        const int tok = p.live_rows[i];
        // ---- S2: combine (max, sumexp) partials of all vocabulary tiles
        float M = -INFINITY;
        for (int n = 0; n < p.num_n; ++n) M = fmaxf(M, p.partials[static_cast<size_t>(n) * p.t_pad + i].x);
        float S = 0.f;
        for (int n = 0; n < p.num_n; ++n) {
            const float2 q = p.partials[static_cast<size_t>(n) * p.t_pad + i];
            S += q.y * expf(q.x - M);
        }
        const float lse = M + logf(S);
        int tmode = p.mode;
        if (p.mode == MODE_MIXED) tmode = (p.mask[tok] == 1) ? MODE_FKL : MODE_MC;
        const int Cr = (p.mode == MODE_MIXED) ? (tmode == MODE_FKL ? p.k_fkl : p.K_mc) : p.C;
        const float* zc = p.zc + static_cast<size_t>(i) * p.C;
        const unsigned char* pm = p.perm + static_cast<size_t>(i) * p.C;
        const float* lam = p.lam + static_cast<size_t>(tok) * p.ld_cache;
        const float* old = p.old ? p.old + static_cast<size_t>(tok) * p.ld_cache : nullptr;
        float* beta = p.beta + static_cast<size_t>(i) * p.C;
        float alpha = 0.f;
        if (tmode == MODE_FKL) {
            float logZq = 0.f, logZp = 0.f;
            if (!(p.flags & FL_NO_RENORM_TEACHER)) {
                float mq = -INFINITY;
                for (int s = 0; s < Cr; ++s) mq = fmaxf(mq, lam[pm[s]]);
                float zq = 0.f;
                for (int s = 0; s < Cr; ++s) zq += expf(lam[pm[s]] - mq);
                logZq = mq + logf(zq);
            }
            if (p.flags & FL_RENORM_STUDENT) {
                float mp = -INFINITY;
                for (int s = 0; s < Cr; ++s) mp = fmaxf(mp, zc[s] - lse);
                float zp = 0.f;
                for (int s = 0; s < Cr; ++s) zp += expf(zc[s] - lse - mp);
                logZp = mp + logf(zp);
            }
            float sq = 0.f;
            for (int s = 0; s < Cr; ++s) sq += expf(lam[pm[s]] - logZq);
            for (int s = 0; s < Cr; ++s) {
                const float l = lam[pm[s]] - logZq;
                const float ell = zc[s] - lse;
                const float qt = expf(l);
                L += qt * (l - (ell - logZp));
                beta[s] = rs * ((p.flags & FL_RENORM_STUDENT) ? sq * expf(ell - logZp) - qt : -qt);
                if (p.slp_out) p.slp_out[static_cast<size_t>(tok) * p.ld_cache + pm[s]] = ell;
            }
            alpha = (p.flags & FL_RENORM_STUDENT) ? 0.f : sq;
        } else if (tmode == MODE_RKL_TOPK) {
            // App. A.1 Eq.(8)-(10) PAPER.md:289-303: KL(p~ || q~), both renormalised on the cached (fixed) support;
            // the full-vocabulary lse cancels and the gradient is purely sparse (alpha = 0).
            float mq = -INFINITY, mp = -INFINITY;
            for (int s = 0; s < Cr; ++s) { mq = fmaxf(mq, lam[pm[s]]); mp = fmaxf(mp, zc[s]); }
            float zq = 0.f, zp = 0.f;
            for (int s = 0; s < Cr; ++s) { zq += expf(lam[pm[s]] - mq); zp += expf(zc[s] - mp); }
            const float logZq = mq + logf(zq), logZp = mp + logf(zp);
            for (int s = 0; s < Cr; ++s) {
                const float lp = zc[s] - logZp, lq = lam[pm[s]] - logZq;
                L += expf(lp) * (lp - lq);
            }
            for (int s = 0; s < Cr; ++s) {
                const float lp = zc[s] - logZp, lq = lam[pm[s]] - logZq;
                beta[s] = rs * expf(lp) * (lp - lq - L);
                if (p.slp_out) p.slp_out[static_cast<size_t>(tok) * p.ld_cache + pm[s]] = zc[s] - lse;
            }
            alpha = 0.f;
        } else {
            const float invm = 1.f / static_cast<float>(Cr);
            float sum_term = 0.f, sum_w = 0.f;
            float sx = 0.f, sxx = 0.f;                      // one-sample estimates X_j = -rho_j A_theta,j (Eq.(16))
            float x_first = 0.f;                            // X of the caller's slot 0 (the one-sample estimator L^MC_1)
            for (int s = 0; s < Cr; ++s) {
                const float ell = zc[s] - lse;
                const float o = old[pm[s]];
                const float lm = lam[pm[s]];
                const float rho = expf(ell - o);
                const float A = (p.flags & FL_SUR_A_OLD) ? (lm - o) : (lm - ell);
                float term = rho * A, w = rho * A;
                if (p.rho_out) p.rho_out[static_cast<size_t>(tok) * p.ld_rho + pm[s]] = rho;
                { const float x = -rho * (lm - ell); sx += x; sxx += x * x; if (pm[s] == 0) x_first = x; }
                if (p.flags & FL_SUR_CLIP) {
                    const float rbar = fminf(fmaxf(rho, 1.f - CLIP_EPS), 1.f + CLIP_EPS);
                    const float cl = rbar * A;
                    const bool active = (term <= cl) || (rbar == rho);
                    w = active ? term : 0.f;
                    term = fminf(term, cl);
                }
                sum_term += term;
                sum_w += w;
                beta[s] = -rs * invm * w;
                if (p.slp_out) p.slp_out[static_cast<size_t>(tok) * p.ld_cache + pm[s]] = ell;
            }
            L = -sum_term * invm;
            alpha = sum_w * invm;
            const float var1 = Cr > 1 ? fmaxf(0.f, (sxx - sx * sx * invm) / static_cast<float>(Cr - 1)) : 0.f;
            if (p.var1_out) p.var1_out[tok] = var1;
            if (p.seq_l1) { p.seq_l1[tok] = x_first; p.seq_var1[tok] = var1; }
        }
        for (int s = Cr; s < p.C; ++s) beta[s] = 0.f;
        p.lse2[i] = lse * LOG2E;
        p.coef[i] = rs * alpha;
        p.per_token_kl[tok] = L;
        if (p.lse_out) p.lse_out[tok] = lse;
    }
    // ---- S5: deterministic block sum (fp64), finished by k_loss_final in block order
    __shared__ double sh[128];
    sh[threadIdx.x] = static_cast<double>(L);
    __syncthreads();
    for (int s = 64; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) p.block_sums[blockIdx.x] = sh[0];
}

__global__ void __launch_bounds__(256) k_loss_final(const double* __restrict__ block_sums, int nblocks, const int* __restrict__ n_live,
                                                    float norm_override, float* __restrict__ loss) {
    __shared__ double sh[256];
    double a = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += 256) a += block_sums[b];
    sh[threadIdx.x] = a;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double norm = norm_override > 0.f ? static_cast<double>(norm_override) : static_cast<double>(*n_live);
        *loss = norm > 0.0 ? static_cast<float>(sh[0] / norm) : 0.f;
    }
}

// Sequence-level diagnostics (opd_set_seq_diagnostics; Eq.(17)): per sequence the timestep averages of
// the m-sample and of the one-sample estimator and the fixed-path variance of the former.  One block per sequence,
// fp64 tree reduction in a fixed order.
__global__ void __launch_bounds__(256) k_seq_diag(const int* __restrict__ cu, int n_seq, int T, const unsigned char* __restrict__ mask,
                                                  int mode, int m, const float* __restrict__ per_token_kl, const float* __restrict__ l1,
                                                  const float* __restrict__ var1, float* __restrict__ mean_m, float* __restrict__ mean_1,
                                                  float* __restrict__ var_m) {
    const int n = blockIdx.x;
    const int b = max(0, min(T, cu[n])), e = max(b, min(T, cu[n + 1]));
    double cnt = 0.0, sm = 0.0, s1 = 0.0, sv = 0.0;
    for (int t = b + threadIdx.x; t < e; t += blockDim.x) {
        const int mk = mask[t];
        if (mk != 0 && (mode == MODE_MC || mk == 2)) { cnt += 1.0; sm += per_token_kl[t]; s1 += l1[t]; sv += var1[t]; }
    }
    __shared__ double sh[4][256];
    sh[0][threadIdx.x] = cnt; sh[1][threadIdx.x] = sm; sh[2][threadIdx.x] = s1; sh[3][threadIdx.x] = sv;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s)
            for (int q = 0; q < 4; ++q) sh[q][threadIdx.x] += sh[q][threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double Tn = sh[0][0];
        mean_m[n] = Tn > 0 ? static_cast<float>(sh[1][0] / Tn) : 0.f;
        mean_1[n] = Tn > 0 ? static_cast<float>(sh[2][0] / Tn) : 0.f;
        var_m[n] = Tn > 0 ? static_cast<float>(sh[3][0] / (Tn * Tn * m)) : 0.f;
    }
}

// gathered logits back in caller slot order (opd_debug_logits)
__global__ void k_unsort_gather(const float* __restrict__ zc, const unsigned char* __restrict__ perm, int T, int C,
                                float* __restrict__ out) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < T * C) {
        const int r = e / C;
        out[static_cast<size_t>(r) * C + perm[e]] = zc[e];
    }
}

}  // namespace opd

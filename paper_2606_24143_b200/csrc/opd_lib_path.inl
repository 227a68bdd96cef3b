// The hot path: S0 pre-pass -> S1-S3 forward GEMM -> S4-S5 estimators -> S6-S8 backward super-tiles.
// Included by opd_lib.cu.

struct PathIO {
    int T, d, V; opd_dtype_t dtype;
    const void* hidden; long ld_hidden;
    const void* W; long ldw_k, ldw_v;
    const int* cache_idx; long ld_cache;
    const float* lam; const float* old;
    const unsigned char* mask;
    opd_mode_t mode; int k_or_K; unsigned flags; float norm_override;
    float* loss; float* per_token_kl; float* lse_out; float* slp_out;
    void* grad_hidden; long ld_gh;
    void* grad_W; long ldgw_k, ldgw_v;
    // debug
    float* dbg_logits; float* dbg_gathered; bool stop_after_fwd; bool all_live;
};

// Launch the persistent backward kernel on as many CTAs (pairs) as can be resident at once on the handle's device (one
// wave).  Tiles are claimed dynamically in dependency order (opd_bwd_kernel.cuh), so the kernel also completes when fewer
// CTAs than that get to run (another kernel holding SMs, MPS, SM-limited contexts): residency is a speed matter only.
template <bool DENSE>
static opd_status_t launch_bwd(opd_handle_s* h, cudaStream_t st, const CUtensorMap& m_xc_k, const CUtensorMap& m_w_fwd,
                               const CUtensorMap& m_gs_k, const CUtensorMap& m_w_dx, const CUtensorMap& m_xc_mn,
                               const CUtensorMap& m_gs_mn, const CUtensorMap& m_tx_k, const CUtensorMap& m_wt_fwd, const BwdParams& bp,
                               const L2Window& win = L2Window{}) {
    int& cached = h->bwd_grid[h->cg][DENSE ? 1 : 0];      // per handle = per device; a failed query is not cached
    if (cached < 1) {
        const int r = h->cg == 2 ? max_resident_groups<2, bwd_stages<2>()>(bwd_kernel<2, DENSE>, h->num_sms, BWD_THREADS)
                                 : max_resident_groups<1, bwd_stages<1>()>(bwd_kernel<1, DENSE>, h->num_sms, BWD_THREADS);
        if (r < 1) OPD_FAIL(h, OPD_ERR_CUDA, "the backward kernel cannot be made resident on device %d", h->device);
        cached = r * h->cg;
    }
    const int grid = cached;
    constexpr int S2 = bwd_stages<2>(), S1 = bwd_stages<1>();
    if (h->cg == 2) OPD_CUDA(h, (launch_cg_w<2, S2>)(bwd_kernel<2, DENSE>, grid, BWD_THREADS, st, win, m_xc_k, m_w_fwd, m_gs_k, m_w_dx, m_xc_mn, m_gs_mn, m_tx_k, m_wt_fwd, bp));
    else OPD_CUDA(h, (launch_cg_w<1, S1>)(bwd_kernel<1, DENSE>, grid, BWD_THREADS, st, win, m_xc_k, m_w_fwd, m_gs_k, m_w_dx, m_xc_mn, m_gs_mn, m_tx_k, m_wt_fwd, bp));
    return OPD_OK;
}

static void phase_mark(opd_handle_s* h, cudaStream_t st, int phase, int end) {
    if (h->phase_events) cudaEventRecord(h->phase_events[2 * phase + end], st);
}

static opd_status_t run_path(opd_handle_s* h, cudaStream_t st, const PathIO& a) {
    if (!h->arch_ok) OPD_FAIL(h, OPD_ERR_ARCH, "device %d is not compute capability 10.x (sm_100a required, no fallback)", h->device);
    const int T = a.T, d = a.d, V = a.V;
    int kf, Km;
    const int C = cache_width(a.mode, a.k_or_K, &kf, &Km);
    if (a.mode != OPD_FKL_TOPK && a.mode != OPD_RKL_MC && a.mode != OPD_MIXED && a.mode != OPD_RKL_TOPK) OPD_FAIL(h, OPD_ERR_BAD_ARG, "unknown mode %d", (int)a.mode);
    if (a.dtype != OPD_BF16 && a.dtype != OPD_FP32) OPD_FAIL(h, OPD_ERR_BAD_ARG, "unknown dtype %d", (int)a.dtype);
    opd_status_t s = check_shape(h, T, d, V, C);
    if (s != OPD_OK) return s;
    if (a.mode == OPD_MIXED && (kf < 1 || Km < 1)) OPD_FAIL(h, OPD_ERR_BAD_SHAPE, "OPD_MIXED needs k>=1 and K>=1 (k_or_K = k | K<<16)");
    const unsigned known = OPD_F_NO_RENORM_TEACHER | OPD_F_RENORM_STUDENT | OPD_F_GRADW_ACCUM | OPD_F_GRADW_BF16 | OPD_F_VALIDATE_IDX |
                           OPD_F_FWD_ONLY | OPD_F_SUR_CLIP | OPD_F_SUR_A_OLD;
    if (a.flags & ~known) OPD_FAIL(h, OPD_ERR_BAD_ARG, "unknown flag bits 0x%x", a.flags & ~known);
    if (h->seq_n > 0 && !a.stop_after_fwd && (a.mode == OPD_RKL_MC || a.mode == OPD_MIXED) && (a.flags & (OPD_F_SUR_CLIP | OPD_F_SUR_A_OLD)))
        OPD_FAIL(h, OPD_ERR_BAD_ARG, "opd_set_seq_diagnostics is on: its outputs describe Eq.(15) (A_theta, unclipped ratio) and cannot be "
                 "combined with OPD_F_SUR_CLIP / OPD_F_SUR_A_OLD (flags 0x%x); switch the hook off for surrogate calls", a.flags);
    const bool fwd_only = (a.flags & OPD_F_FWD_ONLY) || a.stop_after_fwd;
    const bool fp32 = a.dtype == OPD_FP32;
    const int esz = fp32 ? 4 : 2;
    if (!a.hidden || !a.W || !a.cache_idx || (!a.stop_after_fwd && (!a.lam || !a.loss || !a.per_token_kl)))
        OPD_FAIL(h, OPD_ERR_BAD_ARG, "null input/output pointer");
    if (!a.all_live && !a.mask) OPD_FAIL(h, OPD_ERR_BAD_ARG, "mask is null");
    if ((a.mode == OPD_RKL_MC || a.mode == OPD_MIXED) && !a.old && !a.stop_after_fwd) OPD_FAIL(h, OPD_ERR_BAD_ARG, "cache_old_logp is required for RKL_MC / MIXED");
    if (!fwd_only && (!a.grad_hidden || !a.grad_W)) OPD_FAIL(h, OPD_ERR_BAD_ARG, "grad pointers are null (use OPD_F_FWD_ONLY)");
    const int wl = (a.ldw_v == 1) ? 0 : ((a.ldw_k == 1) ? 1 : -1);       // 0: [d,V] row-major, 1: [V,d] row-major
    if (wl < 0) OPD_FAIL(h, OPD_ERR_BAD_ARG, "one of ldw_k / ldw_v must be 1");
    const long ldw = wl == 0 ? a.ldw_k : a.ldw_v;
    if (ldw < (wl == 0 ? V : d)) OPD_FAIL(h, OPD_ERR_BAD_ARG, "W row stride %ld too small", ldw);
    const int al = 16 / esz;
    if ((reinterpret_cast<uintptr_t>(a.hidden) & 15) || (reinterpret_cast<uintptr_t>(a.W) & 15) || a.ld_hidden % al || ldw % al ||
        a.ld_hidden < d)
        OPD_FAIL(h, OPD_ERR_BAD_ARG, "hidden / W must be 16-byte aligned with row strides that are multiples of %d elements", al);
    if (a.ld_cache < C) OPD_FAIL(h, OPD_ERR_BAD_ARG, "ld_cache %ld < C %d", a.ld_cache, C);
    long ldgw = 0;                                 // row stride of the caller's grad_W (elements of ITS dtype)
    const bool gw_bf16 = !fwd_only && (a.flags & OPD_F_GRADW_BF16);
    if (!fwd_only) {
        const int gwl = (a.ldgw_v == 1) ? 0 : ((a.ldgw_k == 1) ? 1 : -1);
        if (gwl != wl && !(wl == 0 && a.ldgw_v == 1) ) OPD_FAIL(h, OPD_ERR_BAD_ARG, "grad_W must use the same unit stride as W");
        ldgw = wl == 0 ? a.ldgw_k : a.ldgw_v;
        if (ldgw < (wl == 0 ? V : d) || ldgw % (gw_bf16 ? 8 : 4) || (reinterpret_cast<uintptr_t>(a.grad_W) & 15))
            OPD_FAIL(h, OPD_ERR_BAD_ARG, "grad_W must be 16-byte aligned, row stride a multiple of %d and >= the inner extent", gw_bf16 ? 8 : 4);
        if (a.ld_gh < d || a.ld_gh % al || (reinterpret_cast<uintptr_t>(a.grad_hidden) & 15))
            OPD_FAIL(h, OPD_ERR_BAD_ARG, "grad_hidden must be 16-byte aligned with a row stride that is a multiple of %d", al);
    }
    if (!get_encode_fn()) OPD_FAIL(h, OPD_ERR_CUDA, "cuTensorMapEncodeTiled not available from the driver");

    OPD_ON_DEVICE(h);
    h->cg = cta_group_setting();
    const uint32_t b_box = BN / h->cg;                    // rows of a K-major B box: each CTA of a pair loads half of N
    const Plan p = make_plan(T, d, V, C, fp32, a.flags | (a.stop_after_fwd ? OPD_F_FWD_ONLY : 0), (int)a.mode);
    s = ensure_workspace(h, p.total, st);
    if (s != OPD_OK) return s;
    h->n_kernels = h->n_gemm = 0;
    h->super_rows = p.Tb; h->super_cols = p.Vb;
    uint8_t* ws = static_cast<uint8_t*>(h->ws);
    int* n_live = reinterpret_cast<int*>(ws + p.off_nlive);
    int* bad_idx = reinterpret_cast<int*>(ws + p.off_badidx);
    int* live_rows = reinterpret_cast<int*>(ws + p.off_live_rows);
    __nv_bfloat16* xc = reinterpret_cast<__nv_bfloat16*>(ws + p.off_xc);
    __nv_bfloat16* wsplit = reinterpret_cast<__nv_bfloat16*>(ws + p.off_wsplit);
    int* sorted_idx = reinterpret_cast<int*>(ws + p.off_sorted);
    unsigned char* perm = ws + p.off_perm;
    float* zc = reinterpret_cast<float*>(ws + p.off_zc);
    float* beta = reinterpret_cast<float*>(ws + p.off_beta);
    float2* partials = reinterpret_cast<float2*>(ws + p.off_partials);
    float* lse2 = reinterpret_cast<float*>(ws + p.off_lse2);
    float* coef = reinterpret_cast<float*>(ws + p.off_coef);
    __nv_bfloat16* gs = reinterpret_cast<__nv_bfloat16*>(ws + p.off_gs);
    float* dxacc = reinterpret_cast<float*>(ws + p.off_dxacc);
    double* block_sums = reinterpret_cast<double*>(ws + p.off_block_sums);
    // fp32 array the backward accumulates grad_W in: the caller's, or (OPD_F_GRADW_BF16) a dense scratch copy that is
    // rounded into the caller's bf16 array at the end (k_emit_bf16)
    const int gw_rows = wl == 0 ? d : V, gw_cols = wl == 0 ? V : d;
    float* gw32 = gw_bf16 ? reinterpret_cast<float*>(ws + p.off_gw32) : static_cast<float*>(a.grad_W);
    const long ldgw32 = gw_bf16 ? gw_cols : ldgw;
    const bool gw_accum = (a.flags & OPD_F_GRADW_ACCUM) && !gw_bf16;     // accumulate INTO gw32 (bf16: the scratch starts fresh)

    // ------------------------------------------------------------------ S0 pre-pass
    phase_mark(h, st, OPD_PHASE_PREP, 0);
    OPD_CUDA(h, cudaMemsetAsync(bad_idx, 0, 4, st));
    OPD_CUDA(h, cudaMemsetAsync(zc, 0, sizeof(float) * (size_t)p.t_pad * C, st));
    if (a.per_token_kl) OPD_CUDA(h, cudaMemsetAsync(a.per_token_kl, 0, sizeof(float) * T, st));
    if (!fwd_only) {
        OPD_CUDA(h, cudaMemset2DAsync(a.grad_hidden, (size_t)a.ld_gh * esz, 0, (size_t)d * esz, T, st));
    }
    k_compact<<<1, 1024, 0, st>>>(a.mask, T, a.all_live ? 1 : 0, live_rows, n_live);
    if (!fwd_only && !gw_accum && !p.sparse_bwd) {
        // An overwriting call needs no memset of grad_W: the grad_W tiles of the first token super-tile store (dense
        // backward; the sparse backward writes every column exactly once).  Only a call without any live token zeroes it.
        k_zero_matrix<<<h->num_sms * 4, 256, 0, st>>>(gw32, ldgw32, gw_rows, gw_cols, n_live);
        h->n_kernels++;
    }
    k_gather_rows<<<p.t_pad, 256, 0, st>>>(a.hidden, a.ld_hidden, fp32 ? 1 : 0, d, p.t_pad, live_rows, n_live, xc, (long)p.xc_plane);
    k_sort_cache<<<ceil_div(T, 8), 256, 0, st>>>(a.cache_idx, a.ld_cache, a.mask, (int)a.mode, kf, Km, C, V, live_rows, n_live,
                                                 sorted_idx, perm, bad_idx);
    h->n_kernels += 3;
    const __nv_bfloat16* wq = static_cast<const __nv_bfloat16*>(a.W);   // bf16 operand planes of W
    long ldwq = ldw;
    size_t wq_plane = 0;
    if (fp32) {
        const int rows = wl == 0 ? d : V, cols = wl == 0 ? V : d;
        k_split_matrix<<<h->num_sms * 8, 256, 0, st>>>(static_cast<const float*>(a.W), ldw, rows, cols, wsplit, (long)p.w_plane);
        h->n_kernels++;
        wq = wsplit; ldwq = cols; wq_plane = p.w_plane;
    }
    OPD_CUDA(h, cudaGetLastError());
    phase_mark(h, st, OPD_PHASE_PREP, 1);

    // ------------------------------------------------------------------ tensor maps
    const uint64_t np = p.planes;
    CUtensorMap m_xc_k, m_xc_mn, m_w_fwd, m_w_dx, m_gs_k, m_gs_mn;
    bool ok = true;
    // Xc [t_pad][d]: K-major A of the logits GEMMs (box 64 x 128); MN-major operand of the grad_W GEMM (box 64 x 64)
    ok &= make_map(&m_xc_k, xc, d, p.t_pad, np, (uint64_t)d * 2, p.xc_plane * 2, BM);
    ok &= make_map(&m_xc_mn, xc, d, p.t_pad, np, (uint64_t)d * 2, p.xc_plane * 2, MN_BOX);
    const uint64_t wplane_b = fp32 ? wq_plane * 2 : (uint64_t)ldwq * 2 * (wl == 0 ? d : V);
    if (wl == 0) {   // W [d][V]: logits B is MN-major (n = v contiguous); dX B is K-major (k = v contiguous)
        ok &= make_map(&m_w_fwd, wq, V, d, np, (uint64_t)ldwq * 2, wplane_b, MN_BOX);
        ok &= make_map(&m_w_dx, wq, V, d, np, (uint64_t)ldwq * 2, wplane_b, b_box);
    } else {         // W [V][d]: logits B is K-major; dX B is MN-major (n = d contiguous, k = v rows)
        ok &= make_map(&m_w_fwd, wq, d, V, np, (uint64_t)ldwq * 2, wplane_b, b_box);
        ok &= make_map(&m_w_dx, wq, d, V, np, (uint64_t)ldwq * 2, wplane_b, MN_BOX);
    }
    if (!fwd_only) {
        ok &= make_map(&m_gs_k, gs, p.Vb, p.Tb, np * p.gs_bufs, (uint64_t)p.Vb * 2, p.gs_plane * 2, BM);
        ok &= make_map(&m_gs_mn, gs, p.Vb, p.Tb, np * p.gs_bufs, (uint64_t)p.Vb * 2, p.gs_plane * 2, MN_BOX);
    }
    DxEpi::Params dxp{};
    DwEpi::Params dwp{};
    if (!fwd_only) {
        ok &= make_map_f32(&dxp.m_acc, dxacc, d, p.Tb, (uint64_t)d * 4);
        ok &= make_map_f32(&dwp.m_gw, gw32, gw_cols, gw_rows, (uint64_t)ldgw32 * 4);
        dxp.acc = dxacc; dxp.ld_acc = d; dxp.out = a.grad_hidden; dxp.ld_out = a.ld_gh; dxp.out_fp32 = fp32 ? 1 : 0;
        dxp.live_rows = live_rows;
        dxp.hint = hint_policy(env_int("OPD_HINT_DX", 0));
        dwp.hint = hint_policy(env_int("OPD_HINT_GW", 0));
#ifdef OPD_EXPERIMENTS
        dxp.dbg = dwp.dbg = env_int("OPD_DBG_ACC", 0);
#endif
    }
    if (!ok) OPD_FAIL(h, OPD_ERR_CUDA, "cuTensorMapEncodeTiled failed");

    // ------------------------------------------------------------------ S1-S3 forward
    phase_mark(h, st, OPD_PHASE_FWD, 0);
    {
        GemmParams gp{};
        gp.M = T; gp.N = V; gp.K = d; gp.num_n = p.num_n;
        gp.group_m = std::max(1, env_int("OPD_GROUP_M", 16));
        gp.a_mn = 0; gp.b_mn = (wl == 0); gp.a_off = 0; gp.b_off = 0; gp.ka_off = 0; gp.kb_off = 0;
        set_segments(gp, p.planes);
        gp.a_hint = hint_policy(env_int("OPD_HINT_FX", 0)); gp.b_hint = hint_policy(env_int("OPD_HINT_FW", 0));
        gp.tok_dim = TOK_M; gp.tok_off = 0; gp.n_live = n_live;
#ifdef OPD_EXPERIMENTS
        gp.skip_b = env_int("OPD_SKIP_B", 0);                 // timing experiment: what the W loads of the forward cost (wrong results)
#endif
        FwdEpi::Params ep{partials, p.t_pad, sorted_idx, zc, C, V, a.dbg_logits};
        OPD_CUDA(h, launch_gemm<FwdEpi>(h, st, m_xc_k, m_w_fwd, gp, ep));
    }
    phase_mark(h, st, OPD_PHASE_FWD, 1);
    if (a.stop_after_fwd) {
        if (a.dbg_gathered) {
            k_unsort_gather<<<ceil_div(T * C, 256), 256, 0, st>>>(zc, perm, T, C, a.dbg_gathered);
            h->n_kernels++;
        }
        OPD_CUDA(h, cudaGetLastError());
        return OPD_OK;
    }

    // ------------------------------------------------------------------ S4-S5 estimators, loss
    phase_mark(h, st, OPD_PHASE_EST, 0);
    {
        EstParams e{};
        e.partials = partials; e.num_n = p.num_n; e.t_pad = p.t_pad; e.zc = zc; e.perm = perm;
        e.lam = a.lam; e.old = a.old; e.ld_cache = a.ld_cache; e.mask = a.mask; e.live_rows = live_rows; e.n_live = n_live;
        e.mode = (int)a.mode; e.k_fkl = kf; e.K_mc = Km; e.C = C; e.flags = a.flags; e.norm_override = a.norm_override;
        e.lse2 = lse2; e.coef = coef; e.beta = beta; e.per_token_kl = a.per_token_kl; e.lse_out = a.lse_out; e.slp_out = a.slp_out;
        e.block_sums = block_sums;
        if ((h->diag_rho || h->diag_var1) && (T > h->diag_rows || (h->diag_rho && C > h->diag_cols)))
            OPD_FAIL(h, OPD_ERR_BAD_ARG, "the diagnostics arrays set with opd_set_diagnostics hold %d x %d entries, this call needs %d x %d",
                     h->diag_rows, h->diag_cols, T, C);
        e.rho_out = h->diag_rho; e.ld_rho = h->diag_ld_rho; e.var1_out = h->diag_var1;
        if (h->diag_var1) OPD_CUDA(h, cudaMemsetAsync(h->diag_var1, 0, sizeof(float) * T, st));
        const bool seq_diag = h->seq_n > 0 && (a.mode == OPD_RKL_MC || a.mode == OPD_MIXED);
        if (seq_diag) { e.seq_l1 = reinterpret_cast<float*>(ws + p.off_seq_l1); e.seq_var1 = reinterpret_cast<float*>(ws + p.off_seq_var1); }
        k_estimator<<<p.est_blocks, 128, 0, st>>>(e);
        if (seq_diag) {
            k_seq_diag<<<h->seq_n, 256, 0, st>>>(h->seq_cu, h->seq_n, T, a.mask, (int)a.mode, Km, a.per_token_kl, e.seq_l1, e.seq_var1,
                                                  h->seq_mean_m, h->seq_mean_1, h->seq_var_m);
            h->n_kernels++;
        }
        k_loss_final<<<1, 256, 0, st>>>(block_sums, p.est_blocks, n_live, a.norm_override, a.loss);
        h->n_kernels += 2;
        OPD_CUDA(h, cudaGetLastError());
    }
    phase_mark(h, st, OPD_PHASE_EST, 1);

    // ------------------------------------------------------------------ S6-S8 backward, super-tile by super-tile
    phase_mark(h, st, OPD_PHASE_BWD, 0);
    // alpha_t == 0 on every row: the gradient lives on the cached columns only, no softmax tile has to be re-formed
    const bool sparse_bwd = p.sparse_bwd;
    if (!fwd_only && sparse_bwd) {
        const void* Wv = a.W;                                   // [V,d] view of W: contiguous d-vectors per column
        long ldwv = ldw;
        if (wl == 0) {
            void* wt = ws + p.off_wt;
            const dim3 tg(ceil_div(V, 32), ceil_div(d, 32));
            if (fp32) k_transpose<float><<<tg, dim3(32, 8), 0, st>>>(static_cast<const float*>(a.W), ldw, d, V, static_cast<float*>(wt), (long)d);
            else k_transpose<__nv_bfloat16><<<tg, dim3(32, 8), 0, st>>>(static_cast<const __nv_bfloat16*>(a.W), ldw, d, V,
                                                                        static_cast<__nv_bfloat16*>(wt), (long)d);
            Wv = wt; ldwv = d;
            h->n_kernels++;
        }
        if (fp32) k_sparse_gh<float><<<p.t_pad, 256, 0, st>>>(Wv, ldwv, d, C, sorted_idx, beta, live_rows, n_live, a.grad_hidden, a.ld_gh);
        else k_sparse_gh<__nv_bfloat16><<<p.t_pad, 256, 0, st>>>(Wv, ldwv, d, C, sorted_idx, beta, live_rows, n_live, a.grad_hidden, a.ld_gh);
        // grad_W: sort the (column, entry) pairs by column (stable), then one block per group of 8 columns
        const size_t N = p.sort_n;
        uint32_t* kbuf[2] = {reinterpret_cast<uint32_t*>(ws + p.off_skeys), reinterpret_cast<uint32_t*>(ws + p.off_skeys) + N};
        uint32_t* vbuf[2] = {kbuf[1] + N, kbuf[1] + 2 * N};
        uint32_t* hist = reinterpret_cast<uint32_t*>(ws + p.off_shist);
        k_sparse_keys<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(sorted_idx, C, N, n_live, V, kbuf[0], vbuf[0]);
        int key_bits = 1;
        while ((1u << key_bits) <= (unsigned)V && key_bits < 32) ++key_bits;                 // keys are in [0, V]
        int cur = 0;
        for (int shift = 0; shift < key_bits; shift += 8, cur ^= 1) {
            k_radix_hist<<<p.sort_blocks, 256, 0, st>>>(kbuf[cur], N, shift, hist, p.sort_blocks);
            k_radix_scan<<<1, 1024, 0, st>>>(hist, (size_t)256 * p.sort_blocks);
            k_radix_scatter<<<p.sort_blocks, 256, 0, st>>>(kbuf[cur], vbuf[cur], N, shift, hist, p.sort_blocks, kbuf[cur ^ 1], vbuf[cur ^ 1]);
            h->n_kernels += 3;
        }
        // hot columns: segments of GW_SEG sorted entries that lie inside one column's run are summed first, all in parallel
        float* part = reinterpret_cast<float*>(ws + p.off_gwseg);
        const dim3 seg_grid((unsigned)(N / GW_SEG), (unsigned)ceil_div(d, GW_KCHUNK));
        if (seg_grid.x) {
            if (fp32) k_sparse_gw_seg<float><<<seg_grid, 256, 0, st>>>(kbuf[cur], vbuf[cur], V, C, beta, live_rows, a.hidden, a.ld_hidden, d, part);
            else k_sparse_gw_seg<__nv_bfloat16><<<seg_grid, 256, 0, st>>>(kbuf[cur], vbuf[cur], V, C, beta, live_rows, a.hidden, a.ld_hidden, d, part);
            h->n_kernels++;
        }
        if (fp32) k_sparse_gw<float><<<V / 8, 256, 0, st>>>(kbuf[cur], vbuf[cur], N, V, C, beta, live_rows, a.hidden, a.ld_hidden, d,
                                                             part, gw32, ldgw32, wl, gw_accum ? 1 : 0);
        else k_sparse_gw<__nv_bfloat16><<<V / 8, 256, 0, st>>>(kbuf[cur], vbuf[cur], N, V, C, beta, live_rows, a.hidden, a.ld_hidden, d,
                                                                part, gw32, ldgw32, wl, gw_accum ? 1 : 0);
        h->n_kernels += 3;
        OPD_CUDA(h, cudaGetLastError());
    }
    if (!fwd_only && !sparse_bwd) {
        // one persistent kernel walks every super-tile: G re-formation, grad_hidden and grad_W tiles interleaved,
        // ordered by dependency counters in global memory (opd_bwd_kernel.cuh)
        int* counters = reinterpret_cast<int*>(ws + p.off_counters);
        OPD_CUDA(h, cudaMemsetAsync(counters, 0, sizeof(int) * (3 * (size_t)p.n_super + 1), st));
        BwdParams bp{};
        bp.d = d; bp.V = V; bp.Tb = p.Tb; bp.Vb = p.Vb; bp.nvb = ceil_div(V, p.Vb); bp.wl = wl; bp.planes = p.planes; bp.gbufs = p.gs_bufs;
        bp.n_live = n_live; bp.g_done = counters; bp.dx_done = counters + p.n_super; bp.dw_done = counters + 2 * p.n_super;
        bp.ticket = counters + 3 * p.n_super;
        bp.dw_store_first = gw_accum ? 0 : 1;
        bp.order = env_int("OPD_BWD_ORDER", 0) & 31;
        bp.q_depth = std::min(SCHED_Q, std::max(1, env_int("OPD_Q_DEPTH", 3)));
        // super-tiles wider than 4096 columns: grad_hidden tiles in groups of 8 row tiles (10 GB fewer G re-reads per C4 launch)
        bp.dx_group = env_int("OPD_DX_GROUP", p.Vb > 4096 ? 8 : 0);
        bp.g = GEpi::Params{gs, p.Tb, (long)p.Vb, (long)p.gs_plane, p.planes, lse2, coef, sorted_idx, beta, C, V, 0ull};
        { const int gh_ = env_int("OPD_HINT_GST", 0); bp.g.st_hint = gh_ ? hint_policy(gh_) : 0ull; }
        bp.dx = dxp;
        bp.dw = dwp;
        bp.hint_x = hint_policy(env_int("OPD_HINT_X", 0)); bp.hint_w = hint_policy(env_int("OPD_HINT_W", 0));
        bp.hint_g = hint_policy(env_int("OPD_HINT_G", 0));
        bp.type_mask = 7;
#ifdef OPD_EXPERIMENTS
        bp.type_mask = env_int("OPD_BWD_TYPES", 7) & 7;       // timing experiment: subsets give wrong gradients
#endif
        // L2 residency experiments: persisting carve-out (device limit) + access-policy window over the G ring / partial sums
        L2Window win{};
        {
            const int pm = env_int("OPD_L2_PERSIST_MB", -1);
            if (pm >= 0) {
                const size_t want = std::min<size_t>((size_t)pm << 20, (size_t)h->l2_persist_max);
                if (want != h->l2_persist) { OPD_CUDA(h, cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, want)); h->l2_persist = want; }
            }
            const int wm = env_int("OPD_L2_WINDOW", 0);
            const size_t gs_b = 2 * p.gs_plane * p.planes * p.gs_bufs, dx_b = sizeof(float) * (size_t)p.Tb * d;
            if (wm == 1) { win.base = gs; win.bytes = gs_b + dx_b; }
            else if (wm == 2) { win.base = gs; win.bytes = gs_b; }
            else if (wm == 3) { win.base = dxacc; win.bytes = dx_b; }
            if (win.bytes) {
                win.bytes = std::min<size_t>(win.bytes, (size_t)h->l2_window_max);
                win.hit_ratio = h->l2_persist ? std::min(1.f, (float)h->l2_persist / (float)win.bytes) : 1.f;
                if (env_int("OPD_L2_VERBOSE", 0))
                    std::fprintf(stderr, "[opd] L2 %d B, persist max %d, window max %d, carve-out %zu, window %zu B hit %.2f\n",
                                 h->l2_bytes, h->l2_persist_max, h->l2_window_max, h->l2_persist, win.bytes, win.hit_ratio);
            }
        }
#ifdef OPD_TRACE
        static unsigned long long* trace_buf = nullptr;     // tracing build: cycle sums per warp role and tile type, printed per call
        if (!trace_buf) OPD_CUDA(h, cudaMalloc(&trace_buf, 128 * 8));
        OPD_CUDA(h, cudaMemsetAsync(trace_buf, 0, 128 * 8, st));
        bp.trace = env_int("OPD_TRACE", 0) ? trace_buf : nullptr;
#endif
        opd_status_t ls = launch_bwd<false>(h, st, m_xc_k, m_w_fwd, m_gs_k, m_w_dx, m_xc_mn, m_gs_mn, m_xc_k, m_w_fwd, bp, win);
        if (ls != OPD_OK) return ls;
#ifdef OPD_TRACE
        if (bp.trace) {
            unsigned long long tb[128];
            OPD_CUDA(h, cudaMemcpyAsync(tb, trace_buf, sizeof(tb), cudaMemcpyDeviceToHost, st));
            OPD_CUDA(h, cudaStreamSynchronize(st));
            static const char* roles[3] = {"mma", "tma", "epi"};
            static const char* types[4] = {"G", "DX", "DW", "Q"};
            std::fprintf(stderr, "[opd trace] kernel cycles summed over CTAs: mma %llu tma %llu epi %llu\n", tb[96], tb[97], tb[98]);
            std::fprintf(stderr, "[opd trace] queue reads (wait / copy / arrive cycles): mma %llu %llu %llu  tma %llu %llu %llu\n",
                         tb[100], tb[101], tb[102], tb[104], tb[105], tb[106]);
            for (int r = 0; r < 3; ++r) for (int ty = 0; ty < 4; ++ty) {
                const unsigned long long* v = tb + (r * 4 + ty) * 8;
                if (!v[0]) continue;
                std::fprintf(stderr, "[opd trace] %s %-2s n=%llu total=%llu s2=%llu s3=%llu s4=%llu s5=%llu s6=%llu s7=%llu\n", roles[r], types[ty],
                             v[0], v[1], v[2], v[3], v[4], v[5], v[6], v[7]);
            }
        }
#endif
        h->n_kernels++; h->n_gemm++;
        OPD_CUDA(h, cudaGetLastError());
    }
    if (gw_bf16) {       // round the fp32 sums into the caller's bf16 grad_W (added to its old contents with OPD_F_GRADW_ACCUM)
        k_emit_bf16<<<h->num_sms * 8, 256, 0, st>>>(gw32, ldgw32, gw_rows, gw_cols, static_cast<__nv_bfloat16*>(a.grad_W), ldgw,
                                                     (a.flags & OPD_F_GRADW_ACCUM) ? 1 : 0);
        h->n_kernels++;
        OPD_CUDA(h, cudaGetLastError());
    }
    phase_mark(h, st, OPD_PHASE_BWD, 1);

    if (a.flags & OPD_F_VALIDATE_IDX) {
        int bad = 0;
        OPD_CUDA(h, cudaMemcpyAsync(&bad, bad_idx, 4, cudaMemcpyDeviceToHost, st));
        OPD_CUDA(h, cudaStreamSynchronize(st));
        if (bad) OPD_FAIL(h, OPD_ERR_BAD_INDEX, "a cache index of a live row is outside [0, %d)", V);
    }
    return OPD_OK;
}

extern "C" opd_status_t opd_loss_fwd_bwd(opd_handle_t h, void* cuda_stream, int T, int d, int V, opd_dtype_t dtype,
    const void* hidden, long ld_hidden, const void* W, long ldw_k, long ldw_v, const int* cache_idx, long ld_cache,
    const float* cache_teacher_logp, const float* cache_old_logp, const unsigned char* mask, opd_mode_t mode, int k_or_K,
    unsigned flags, float norm_override, float* loss, float* per_token_kl, float* lse_out, float* student_logp_out,
    void* grad_hidden, long ld_gh, void* grad_W, long ldgw_k, long ldgw_v) {
    if (!h) return OPD_ERR_BAD_ARG;
    PathIO a{T, d, V, dtype, hidden, ld_hidden, W, ldw_k, ldw_v, cache_idx, ld_cache, cache_teacher_logp, cache_old_logp, mask,
             mode, k_or_K, flags, norm_override, loss, per_token_kl, lse_out, student_logp_out, grad_hidden, ld_gh,
             grad_W, ldgw_k, ldgw_v, nullptr, nullptr, false, false};
    return run_path(h, static_cast<cudaStream_t>(cuda_stream), a);
}

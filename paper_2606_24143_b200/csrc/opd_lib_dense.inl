// opd_dense_kl_fwd_bwd (include/opd.h): dense full-vocabulary forward KL with the teacher's logits recomputed from
// transmitted teacher hidden states (opd_dense.cuh).  Included by opd_lib.cu.

struct DensePlan {
    Plan base;                 // the learner path's plan (student operands, G ring, partial sums, counters ...)
    size_t off_txc, off_wtsplit, off_qring, off_lse_p, off_lse_t, off_lse2_t, off_acc_a, off_acc_b, off_lt, off_qdone, total;
    size_t txc_plane, wt_plane, q_buf_bytes;
};

static DensePlan make_dense_plan(int T, int d, int dT, int V, int fp32, unsigned flags) {
    DensePlan p{};
    p.base = make_plan(T, d, V, 1, fp32, flags, OPD_RKL_MC);
    size_t o = p.base.total;
    auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes, 1024); return r; };
    const int planes = p.base.planes;
    p.txc_plane = (size_t)p.base.t_pad * dT;
    p.off_txc = take(2 * p.txc_plane * planes);
    p.wt_plane = (size_t)dT * V;
    p.off_wtsplit = take(fp32 ? 2 * p.wt_plane * 3 : 0);
    const bool q32 = fp32 || (flags & OPD_F_DENSE_REVERSE);      // the reverse direction keeps log q, always in fp32
    p.q_buf_bytes = align_up((size_t)p.base.Tb * p.base.Vb * (q32 ? 4 : 2), 1024);
    p.off_qring = take(2 * p.q_buf_bytes);
    p.off_lse_p = take(sizeof(float) * (size_t)p.base.t_pad);
    p.off_lse_t = take(sizeof(float) * (size_t)p.base.t_pad);
    p.off_lse2_t = take(sizeof(float) * (size_t)p.base.t_pad);
    p.off_acc_a = take(sizeof(float) * (size_t)p.base.t_pad);
    p.off_acc_b = take(sizeof(float) * (size_t)p.base.t_pad);
    p.off_lt = take(sizeof(float) * (size_t)p.base.t_pad);
    p.off_qdone = take(sizeof(int) * (4 * (size_t)p.base.n_super + 1));      // q_done, g_done, dx_done, dw_done, tile ticket
    p.total = o;
    return p;
}

extern "C" size_t opd_dense_kl_workspace_bytes(int T, int d, int dT, int V, opd_dtype_t dtype, unsigned flags) {
    if (T < 1 || d < 64 || dT < 64 || V < 256) return 0;
    return make_dense_plan(T, d, dT, V, dtype == OPD_FP32, flags).total;
}

extern "C" opd_status_t opd_dense_kl_fwd_bwd(opd_handle_t h, void* cuda_stream, int T, int d, int dT, int V, opd_dtype_t dtype,
    const void* hidden, long ld_hidden, const void* W, long ldw_k, long ldw_v,
    const void* teacher_hidden, long ld_th, const void* W_T, long ldt_k, long ldt_v,
    const unsigned char* mask, unsigned flags, float norm_override,
    float* loss, float* per_token_kl, void* grad_hidden, long ld_gh, void* grad_W, long ldgw_k, long ldgw_v) {
    if (!h) return OPD_ERR_BAD_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (!h->arch_ok) OPD_FAIL(h, OPD_ERR_ARCH, "device %d is not compute capability 10.x (sm_100a required, no fallback)", h->device);
    if (dtype != OPD_BF16 && dtype != OPD_FP32) OPD_FAIL(h, OPD_ERR_BAD_ARG, "unknown dtype %d", (int)dtype);
    if (flags & ~(unsigned)(OPD_F_GRADW_ACCUM | OPD_F_FWD_ONLY | OPD_F_DENSE_REVERSE)) OPD_FAIL(h, OPD_ERR_BAD_ARG, "unsupported flag bits 0x%x", flags);
    const bool reverse = (flags & OPD_F_DENSE_REVERSE) != 0;
    const bool q32 = dtype == OPD_FP32 || reverse;
    opd_status_t s = check_shape(h, T, d, V, 1);
    if (s != OPD_OK) return s;
    if (dT < 64 || dT > 16384 || dT % 64) OPD_FAIL(h, OPD_ERR_BAD_SHAPE, "teacher width dT=%d must be a multiple of 64 in [64,16384]", dT);
    const bool fwd_only = (flags & OPD_F_FWD_ONLY) != 0;
    const bool fp32 = dtype == OPD_FP32;
    const int esz = fp32 ? 4 : 2, al = 16 / esz;
    if (!hidden || !W || !teacher_hidden || !W_T || !mask || !loss || !per_token_kl) OPD_FAIL(h, OPD_ERR_BAD_ARG, "null input/output pointer");
    if (!fwd_only && (!grad_hidden || !grad_W)) OPD_FAIL(h, OPD_ERR_BAD_ARG, "grad pointers are null (use OPD_F_FWD_ONLY)");
    const int wl = (ldw_v == 1) ? 0 : ((ldw_k == 1) ? 1 : -1);
    const int wlt = (ldt_v == 1) ? 0 : ((ldt_k == 1) ? 1 : -1);
    if (wl < 0 || wlt < 0) OPD_FAIL(h, OPD_ERR_BAD_ARG, "one stride of W and of W_T must be 1");
    const long ldw = wl == 0 ? ldw_k : ldw_v, ldwt = wlt == 0 ? ldt_k : ldt_v;
    auto mis = [](const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15) != 0; };
    if (ldw < (wl == 0 ? V : d) || ldwt < (wlt == 0 ? V : dT) || mis(hidden) || mis(W) || mis(teacher_hidden) || mis(W_T) ||
        ld_hidden % al || ld_th % al || ldw % al || ldwt % al || ld_hidden < d || ld_th < dT)
        OPD_FAIL(h, OPD_ERR_BAD_ARG, "operands must be 16-byte aligned with row strides that are multiples of %d elements", al);
    long ldgw = 0;
    if (!fwd_only) {
        if ((wl == 0 ? ldgw_v : ldgw_k) != 1) OPD_FAIL(h, OPD_ERR_BAD_ARG, "grad_W must use the same unit stride as W");
        ldgw = wl == 0 ? ldgw_k : ldgw_v;
        if (ldgw < (wl == 0 ? V : d) || ldgw % 4 || mis(grad_W) || ld_gh < d || ld_gh % al || mis(grad_hidden))
            OPD_FAIL(h, OPD_ERR_BAD_ARG, "grad_hidden / grad_W alignment or strides");
    }
    if (!get_encode_fn()) OPD_FAIL(h, OPD_ERR_CUDA, "cuTensorMapEncodeTiled not available from the driver");

    OPD_ON_DEVICE(h);
    h->cg = cta_group_setting();
    const uint32_t b_box = BN / h->cg;
    const DensePlan dp = make_dense_plan(T, d, dT, V, fp32, flags);
    const Plan& p = dp.base;
    s = ensure_workspace(h, dp.total, st);
    if (s != OPD_OK) return s;
    h->n_kernels = h->n_gemm = 0;
    h->super_rows = p.Tb; h->super_cols = p.Vb;
    uint8_t* ws = static_cast<uint8_t*>(h->ws);
    int* n_live = reinterpret_cast<int*>(ws + p.off_nlive);
    int* live_rows = reinterpret_cast<int*>(ws + p.off_live_rows);
    __nv_bfloat16* xc = reinterpret_cast<__nv_bfloat16*>(ws + p.off_xc);
    __nv_bfloat16* wsplit = reinterpret_cast<__nv_bfloat16*>(ws + p.off_wsplit);
    __nv_bfloat16* txc = reinterpret_cast<__nv_bfloat16*>(ws + dp.off_txc);
    __nv_bfloat16* wtsplit = reinterpret_cast<__nv_bfloat16*>(ws + dp.off_wtsplit);
    float2* partials = reinterpret_cast<float2*>(ws + p.off_partials);
    float* lse2_p = reinterpret_cast<float*>(ws + p.off_lse2);
    float* coef = reinterpret_cast<float*>(ws + p.off_coef);
    float* lse_p = reinterpret_cast<float*>(ws + dp.off_lse_p);
    float* lse_t = reinterpret_cast<float*>(ws + dp.off_lse_t);
    float* lse2_t = reinterpret_cast<float*>(ws + dp.off_lse2_t);
    float* acc_a = reinterpret_cast<float*>(ws + dp.off_acc_a);
    float* acc_b = reinterpret_cast<float*>(ws + dp.off_acc_b);
    float* lt = reinterpret_cast<float*>(ws + dp.off_lt);
    __nv_bfloat16* gs = reinterpret_cast<__nv_bfloat16*>(ws + p.off_gs);
    float* dxacc = reinterpret_cast<float*>(ws + p.off_dxacc);
    double* block_sums = reinterpret_cast<double*>(ws + p.off_block_sums);
    uint8_t* qring = ws + dp.off_qring;

    // ---- pre-pass: compaction of both hidden arrays, fp32 operands split into bf16 planes
    OPD_CUDA(h, cudaMemsetAsync(per_token_kl, 0, sizeof(float) * T, st));
    if (!fwd_only) {
        OPD_CUDA(h, cudaMemset2DAsync(grad_hidden, (size_t)ld_gh * esz, 0, (size_t)d * esz, T, st));
    }
    k_compact<<<1, 1024, 0, st>>>(mask, T, 0, live_rows, n_live);
    if (!fwd_only && !(flags & OPD_F_GRADW_ACCUM)) {       // the first token super-tile stores grad_W; zeros only if no token is live
        k_zero_matrix<<<h->num_sms * 4, 256, 0, st>>>(static_cast<float*>(grad_W), ldgw, wl == 0 ? d : V, wl == 0 ? V : d, n_live);
        h->n_kernels++;
    }
    k_gather_rows<<<p.t_pad, 256, 0, st>>>(hidden, ld_hidden, fp32 ? 1 : 0, d, p.t_pad, live_rows, n_live, xc, (long)p.xc_plane);
    k_gather_rows<<<p.t_pad, 256, 0, st>>>(teacher_hidden, ld_th, fp32 ? 1 : 0, dT, p.t_pad, live_rows, n_live, txc, (long)dp.txc_plane);
    h->n_kernels += 3;
    const __nv_bfloat16 *wq = static_cast<const __nv_bfloat16*>(W), *wtq = static_cast<const __nv_bfloat16*>(W_T);
    long ldwq = ldw, ldwtq = ldwt;
    if (fp32) {
        k_split_matrix<<<h->num_sms * 8, 256, 0, st>>>(static_cast<const float*>(W), ldw, wl == 0 ? d : V, wl == 0 ? V : d, wsplit, (long)p.w_plane);
        k_split_matrix<<<h->num_sms * 8, 256, 0, st>>>(static_cast<const float*>(W_T), ldwt, wlt == 0 ? dT : V, wlt == 0 ? V : dT, wtsplit, (long)dp.wt_plane);
        h->n_kernels += 2;
        wq = wsplit; ldwq = wl == 0 ? V : d;
        wtq = wtsplit; ldwtq = wlt == 0 ? V : dT;
    }
    OPD_CUDA(h, cudaGetLastError());

    // ---- tensor maps
    const uint64_t np = p.planes;
    CUtensorMap m_xc_k, m_xc_mn, m_w_fwd, m_w_dx, m_gs_k, m_gs_mn, m_tx_k, m_wt_fwd;
    bool ok = true;
    ok &= make_map(&m_xc_k, xc, d, p.t_pad, np, (uint64_t)d * 2, p.xc_plane * 2, BM);
    ok &= make_map(&m_xc_mn, xc, d, p.t_pad, np, (uint64_t)d * 2, p.xc_plane * 2, MN_BOX);
    ok &= make_map(&m_tx_k, txc, dT, p.t_pad, np, (uint64_t)dT * 2, dp.txc_plane * 2, BM);
    const uint64_t wplane_b = fp32 ? p.w_plane * 2 : (uint64_t)ldwq * 2 * (wl == 0 ? d : V);
    const uint64_t wtplane_b = fp32 ? dp.wt_plane * 2 : (uint64_t)ldwtq * 2 * (wlt == 0 ? dT : V);
    if (wl == 0) {
        ok &= make_map(&m_w_fwd, wq, V, d, np, (uint64_t)ldwq * 2, wplane_b, MN_BOX);
        ok &= make_map(&m_w_dx, wq, V, d, np, (uint64_t)ldwq * 2, wplane_b, b_box);
    } else {
        ok &= make_map(&m_w_fwd, wq, d, V, np, (uint64_t)ldwq * 2, wplane_b, b_box);
        ok &= make_map(&m_w_dx, wq, d, V, np, (uint64_t)ldwq * 2, wplane_b, MN_BOX);
    }
    if (wlt == 0) ok &= make_map(&m_wt_fwd, wtq, V, dT, np, (uint64_t)ldwtq * 2, wtplane_b, MN_BOX);
    else ok &= make_map(&m_wt_fwd, wtq, dT, V, np, (uint64_t)ldwtq * 2, wtplane_b, b_box);
    ok &= make_map(&m_gs_k, gs, p.Vb, p.Tb, np * p.gs_bufs, (uint64_t)p.Vb * 2, p.gs_plane * 2, BM);
    ok &= make_map(&m_gs_mn, gs, p.Vb, p.Tb, np * p.gs_bufs, (uint64_t)p.Vb * 2, p.gs_plane * 2, MN_BOX);
    DxEpi::Params dxp{};
    DwEpi::Params dwp{};
    if (!fwd_only) {
        ok &= make_map_f32(&dxp.m_acc, dxacc, d, p.Tb, (uint64_t)d * 4);
        ok &= make_map_f32(&dwp.m_gw, grad_W, wl == 0 ? V : d, wl == 0 ? d : V, (uint64_t)ldgw * 4);
        dxp.acc = dxacc; dxp.ld_acc = d; dxp.out = grad_hidden; dxp.ld_out = ld_gh; dxp.out_fp32 = fp32 ? 1 : 0;
        dxp.live_rows = live_rows;
        dxp.hint = dwp.hint = L2_EVICT_NORMAL;
    }
    if (!ok) OPD_FAIL(h, OPD_ERR_CUDA, "cuTensorMapEncodeTiled failed");

    // ---- pass A: lse of both heads (the learner path's forward kernel, no cache to gather)
    GemmParams gp{};
    gp.M = T; gp.N = V; gp.num_n = p.num_n;
    gp.group_m = std::max(1, env_int("OPD_GROUP_M", 16));
    gp.a_mn = 0;
    set_segments(gp, p.planes);
    gp.tok_dim = TOK_M; gp.tok_off = 0; gp.n_live = n_live;
    FwdEpi::Params fep{partials, p.t_pad, nullptr, nullptr, 0, V, nullptr};
    gp.K = d; gp.b_mn = (wl == 0);
    OPD_CUDA(h, launch_gemm<FwdEpi>(h, st, m_xc_k, m_w_fwd, gp, fep));
    k_lse_theta<<<ceil_div(p.t_pad, 8), 256, 0, st>>>(partials, p.num_n, p.t_pad, p.t_pad, 0, lse_p, nullptr);
    gp.K = dT; gp.b_mn = (wlt == 0);
    OPD_CUDA(h, launch_gemm<FwdEpi>(h, st, m_tx_k, m_wt_fwd, gp, fep));
    k_lse_theta<<<ceil_div(p.t_pad, 8), 256, 0, st>>>(partials, p.num_n, p.t_pad, p.t_pad, 0, lse_t, nullptr);
    k_dense_rows<<<ceil_div(p.t_pad, 256), 256, 0, st>>>(lse_p, lse_t, n_live, norm_override, p.t_pad, lse2_p, lse2_t, coef, acc_a, acc_b);
    h->n_kernels += 3;

    // ---- pass B: Q / G (/ grad_hidden / grad_W) tiles in one persistent launch (two launches for the reverse direction)
    int* q_done = reinterpret_cast<int*>(ws + dp.off_qdone);
    int* counters = q_done + p.n_super;
    BwdParams bp{};
    bp.d = d; bp.V = V; bp.Tb = p.Tb; bp.Vb = p.Vb; bp.nvb = ceil_div(V, p.Vb); bp.wl = wl; bp.planes = p.planes; bp.gbufs = p.gs_bufs;
    bp.n_live = n_live; bp.g_done = counters; bp.dx_done = counters + p.n_super; bp.dw_done = counters + 2 * p.n_super; bp.q_done = q_done;
    bp.ticket = counters + 3 * p.n_super;
    bp.dw_store_first = (flags & OPD_F_GRADW_ACCUM) ? 0 : 1;
    bp.dx_group = p.Vb > 4096 ? 8 : 0;
    bp.q_depth = std::min(SCHED_Q, std::max(1, env_int("OPD_Q_DEPTH", 3)));
    bp.dx = dxp; bp.dw = dwp;
    bp.hint_x = bp.hint_w = bp.hint_g = L2_EVICT_NORMAL;
    bp.dT = dT; bp.wl_t = wlt; bp.qbytes = q32 ? 4 : 2; bp.q_buf_bytes = dp.q_buf_bytes;
    bp.q = QEpi::Params{qring, p.Tb, (long)p.Vb, q32 ? 1 : 0, lse2_t, acc_a, V, reverse ? 1 : 0};
    bp.gd = GDenseEpi::Params{gs, p.Tb, (long)p.Vb, (long)p.gs_plane, p.planes, qring, (long)p.Vb, q32 ? 1 : 0, lse2_p, coef, acc_b, V,
                              reverse ? 1 : 0, nullptr};
    const int fwd_types = (1 << T_Q) | (1 << T_G);
    auto launch = [&](int type_mask) -> opd_status_t {
        OPD_CUDA(h, cudaMemsetAsync(q_done, 0, sizeof(int) * (4 * (size_t)p.n_super + 1), st));
        bp.type_mask = type_mask;
        opd_status_t ls = launch_bwd<true>(h, st, m_xc_k, m_w_fwd, m_gs_k, m_w_dx, m_xc_mn, m_gs_mn, m_tx_k, m_wt_fwd, bp);
        if (ls == OPD_OK) { h->n_kernels++; h->n_gemm++; }
        return ls;
    };
    auto loss_kernels = [&]() {
        k_dense_loss<<<p.est_blocks, 128, 0, st>>>(acc_a, acc_b, reverse ? 1 : 0, live_rows, n_live, per_token_kl, reverse ? lt : nullptr, block_sums);
        k_loss_final<<<1, 256, 0, st>>>(block_sums, p.est_blocks, n_live, norm_override, loss);
        h->n_kernels += 2;
    };
    if (!reverse) {
        s = launch(fwd_only ? fwd_types : 15);
        if (s != OPD_OK) return s;
        loss_kernels();                                   // L_t = A_t - B_t, token mean
    } else {
        s = launch(fwd_types);                            // L_t = sum_v p (log p - log q): the gradient tiles need it
        if (s != OPD_OK) return s;
        loss_kernels();
        if (!fwd_only) {
            bp.gd.acc_b = nullptr; bp.gd.lt = lt;
            s = launch(15);
            if (s != OPD_OK) return s;
        }
    }
    OPD_CUDA(h, cudaGetLastError());
    return OPD_OK;
}

// Cache producers: opd_cache_topk / opd_cache_sample (include/opd.h).  Included by opd_lib.cu.
// Pass A = the learner path's forward kernel (per-tile LSE partials), pass B = the same contraction with a
// collecting / sampling epilogue (opd_producer.cuh).

struct ProducerPlan {
    int t_pad, num_n, planes, cap;
    size_t off_nlive, off_live_rows, off_xc, off_wsplit, off_partials, off_lse, off_theta, off_count, off_cand, off_overflow,
           off_tile, off_res, off_perm, total;
    size_t xc_plane, w_plane;
};

static int topk_cap(int V, int k) {
    // candidates per row: elements >= the k-th largest tile maximum; all V columns when there are fewer than k tiles
    return ceil_div(V, BN) < k ? ceil_div(V, 32) * 32 : std::max(4 * k, 256);
}

static ProducerPlan make_producer_plan(int T, int d, int V, int fp32, int k_top, int K_samp) {
    ProducerPlan p{};
    const int TM = BM * cta_group_setting();
    p.t_pad = ceil_div(T, TM) * TM;
    p.num_n = ceil_div(V, BN);
    p.planes = fp32 ? 3 : 1;
    p.cap = k_top > 0 ? topk_cap(V, k_top) : 0;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes, 1024); return r; };
    p.off_nlive = take(4);
    p.off_overflow = take(4);
    p.off_live_rows = take(sizeof(int) * (size_t)p.t_pad);
    p.xc_plane = (size_t)p.t_pad * d;
    p.off_xc = take(2 * p.xc_plane * p.planes);
    p.w_plane = (size_t)d * V;
    p.off_wsplit = take(fp32 ? 2 * p.w_plane * 3 : 0);
    p.off_partials = take(sizeof(float2) * (size_t)p.num_n * p.t_pad);
    p.off_lse = take(sizeof(float) * (size_t)p.t_pad);
    p.off_theta = take(sizeof(float) * (size_t)p.t_pad);
    p.off_count = take(sizeof(int) * (size_t)p.t_pad);
    p.off_cand = take(sizeof(float2) * (size_t)p.t_pad * p.cap);
    p.off_tile = take(sizeof(int) * (size_t)p.t_pad * K_samp);
    p.off_res = take(sizeof(float) * (size_t)p.t_pad * K_samp);
    p.off_perm = take((size_t)p.t_pad * K_samp);
    p.total = o;
    return p;
}

extern "C" size_t opd_cache_workspace_bytes(int T, int d, int V, opd_dtype_t dtype, int k_top, int K_samples) {
    if (T < 1 || d < 64 || V < 256 || k_top < 0 || K_samples < 0 || k_top > 64 || K_samples > 64) return 0;
    return make_producer_plan(T, d, V, dtype == OPD_FP32, k_top, K_samples).total;
}

// which = 0: top-k (n = k), which = 1: samples (n = K, u = uniforms)
static opd_status_t run_producer(opd_handle_s* h, cudaStream_t st, int which, int T, int d, int V, opd_dtype_t dtype,
                                 const void* hidden, long ld_hidden, const void* W, long ldw_k, long ldw_v, const unsigned char* mask, int n,
                                 const float* u, long ld_u, int* idx_out, long ld_idx, float* logp_out, long ld_logp, float* lse_out) {
    if (!h->arch_ok) OPD_FAIL(h, OPD_ERR_ARCH, "device %d is not compute capability 10.x (sm_100a required, no fallback)", h->device);
    if (dtype != OPD_BF16 && dtype != OPD_FP32) OPD_FAIL(h, OPD_ERR_BAD_ARG, "unknown dtype %d", (int)dtype);
    opd_status_t s = check_shape(h, T, d, V, n);
    if (s != OPD_OK) return s;
    if (!hidden || !W || !idx_out || !logp_out || (which == 1 && !u)) OPD_FAIL(h, OPD_ERR_BAD_ARG, "null input/output pointer");
    if (which == 0 && n > V) OPD_FAIL(h, OPD_ERR_BAD_SHAPE, "k=%d exceeds V=%d", n, V);
    const bool fp32 = dtype == OPD_FP32;
    const int esz = fp32 ? 4 : 2;
    const int wl = (ldw_v == 1) ? 0 : ((ldw_k == 1) ? 1 : -1);
    if (wl < 0) OPD_FAIL(h, OPD_ERR_BAD_ARG, "one of ldw_k / ldw_v must be 1");
    const long ldw = wl == 0 ? ldw_k : ldw_v;
    const int al = 16 / esz;
    if (ldw < (wl == 0 ? V : d) || (reinterpret_cast<uintptr_t>(hidden) & 15) || (reinterpret_cast<uintptr_t>(W) & 15) ||
        ld_hidden % al || ldw % al || ld_hidden < d)
        OPD_FAIL(h, OPD_ERR_BAD_ARG, "hidden / W must be 16-byte aligned with row strides that are multiples of %d elements", al);
    if (ld_idx < n || ld_logp < n || (which == 1 && ld_u < n)) OPD_FAIL(h, OPD_ERR_BAD_ARG, "output / uniform row stride smaller than %d", n);
    if (!get_encode_fn()) OPD_FAIL(h, OPD_ERR_CUDA, "cuTensorMapEncodeTiled not available from the driver");

    OPD_ON_DEVICE(h);
    h->cg = cta_group_setting();
    const uint32_t b_box = BN / h->cg;
    const ProducerPlan p = make_producer_plan(T, d, V, fp32, which == 0 ? n : 0, which == 1 ? n : 0);
    s = ensure_workspace(h, p.total, st);
    if (s != OPD_OK) return s;
    h->n_kernels = h->n_gemm = 0;
    uint8_t* ws = static_cast<uint8_t*>(h->ws);
    int* n_live = reinterpret_cast<int*>(ws + p.off_nlive);
    int* overflow = reinterpret_cast<int*>(ws + p.off_overflow);
    int* live_rows = reinterpret_cast<int*>(ws + p.off_live_rows);
    __nv_bfloat16* xc = reinterpret_cast<__nv_bfloat16*>(ws + p.off_xc);
    __nv_bfloat16* wsplit = reinterpret_cast<__nv_bfloat16*>(ws + p.off_wsplit);
    float2* partials = reinterpret_cast<float2*>(ws + p.off_partials);
    float* lse = reinterpret_cast<float*>(ws + p.off_lse);
    float* theta = reinterpret_cast<float*>(ws + p.off_theta);
    int* count = reinterpret_cast<int*>(ws + p.off_count);
    float2* cand = reinterpret_cast<float2*>(ws + p.off_cand);
    int* tgt_tile = reinterpret_cast<int*>(ws + p.off_tile);
    float* tgt_res = reinterpret_cast<float*>(ws + p.off_res);
    unsigned char* perm = ws + p.off_perm;

    // operand staging: rows with mask == 0 are not scored (mask == NULL: every row is)
    OPD_CUDA(h, cudaMemsetAsync(overflow, 0, 4, st));
    k_compact<<<1, 1024, 0, st>>>(mask, T, mask ? 0 : 1, live_rows, n_live);
    k_gather_rows<<<p.t_pad, 256, 0, st>>>(hidden, ld_hidden, fp32 ? 1 : 0, d, p.t_pad, live_rows, n_live, xc, (long)p.xc_plane);
    h->n_kernels += 2;
    const __nv_bfloat16* wq = static_cast<const __nv_bfloat16*>(W);
    long ldwq = ldw;
    size_t wq_plane = 0;
    if (fp32) {
        const int rows = wl == 0 ? d : V, cols = wl == 0 ? V : d;
        k_split_matrix<<<h->num_sms * 8, 256, 0, st>>>(static_cast<const float*>(W), ldw, rows, cols, wsplit, (long)p.w_plane);
        h->n_kernels++;
        wq = wsplit; ldwq = cols; wq_plane = p.w_plane;
    }
    OPD_CUDA(h, cudaGetLastError());
    const uint64_t np = p.planes;
    CUtensorMap m_xc_k, m_w_fwd;
    bool ok = make_map(&m_xc_k, xc, d, p.t_pad, np, (uint64_t)d * 2, p.xc_plane * 2, BM);
    const uint64_t wplane_b = fp32 ? wq_plane * 2 : (uint64_t)ldwq * 2 * (wl == 0 ? d : V);
    if (wl == 0) ok &= make_map(&m_w_fwd, wq, V, d, np, (uint64_t)ldwq * 2, wplane_b, MN_BOX);
    else ok &= make_map(&m_w_fwd, wq, d, V, np, (uint64_t)ldwq * 2, wplane_b, b_box);
    if (!ok) OPD_FAIL(h, OPD_ERR_CUDA, "cuTensorMapEncodeTiled failed");

    GemmParams gp{};
    gp.M = T; gp.N = V; gp.K = d; gp.num_n = p.num_n;
    gp.group_m = std::max(1, env_int("OPD_GROUP_M", 16));
    gp.a_mn = 0; gp.b_mn = (wl == 0);
    set_segments(gp, p.planes);
    gp.tok_dim = TOK_M; gp.tok_off = 0; gp.n_live = n_live;
    {   // pass A: per-tile (max, sum exp) partials
        FwdEpi::Params ep{partials, p.t_pad, nullptr, nullptr, 0, V, nullptr};
        OPD_CUDA(h, launch_gemm<FwdEpi>(h, st, m_xc_k, m_w_fwd, gp, ep));
    }
    k_lse_theta<<<ceil_div(T, 8), 256, 0, st>>>(partials, p.num_n, p.t_pad, T, n, lse, which == 0 ? theta : nullptr);
    h->n_kernels++;
    if (which == 0) {
        OPD_CUDA(h, cudaMemsetAsync(count, 0, sizeof(int) * (size_t)T, st));
        CollectEpi::Params ep{theta, count, cand, p.cap, V};
        OPD_CUDA(h, launch_gemm<CollectEpi>(h, st, m_xc_k, m_w_fwd, gp, ep));
        k_topk_select<<<ceil_div(T, 8), 256, 0, st>>>(cand, count, p.cap, T, n, lse, live_rows, n_live, idx_out, ld_idx, logp_out, ld_logp, overflow);
        h->n_kernels++;
    } else {
        k_sample_targets<<<ceil_div(T, 128), 128, 0, st>>>(partials, p.num_n, p.t_pad, T, n, lse, live_rows, n_live, u, ld_u, tgt_tile, tgt_res, perm);
        SampleEpi::Params ep{tgt_tile, tgt_res, perm, lse, n, V, idx_out, ld_idx, logp_out, ld_logp, live_rows};
        OPD_CUDA(h, launch_gemm<SampleEpi>(h, st, m_xc_k, m_w_fwd, gp, ep));
        h->n_kernels++;
    }
    if (lse_out) { k_scatter_rows_f32<<<ceil_div(T, 256), 256, 0, st>>>(lse, live_rows, n_live, T, lse_out); h->n_kernels++; }
    OPD_CUDA(h, cudaGetLastError());
    if (which == 0) {   // candidate-list overflow (more than `cap` logits tie at / exceed the threshold) is an error, not a silent truncation
        int ov = 0;
        OPD_CUDA(h, cudaMemcpyAsync(&ov, overflow, 4, cudaMemcpyDeviceToHost, st));
        OPD_CUDA(h, cudaStreamSynchronize(st));
        if (ov) OPD_FAIL(h, OPD_ERR_WORKSPACE, "top-k candidate list overflow: a row has %d logits >= its threshold, capacity %d "
                                               "(massively tied logits)", ov, p.cap);
    }
    return OPD_OK;
}

extern "C" opd_status_t opd_cache_topk(opd_handle_t h, void* cuda_stream, int T, int d, int V, opd_dtype_t dtype,
    const void* hidden, long ld_hidden, const void* W, long ldw_k, long ldw_v, const unsigned char* mask, int k,
    int* idx_out, long ld_idx, float* logp_out, long ld_logp, float* lse_out) {
    if (!h) return OPD_ERR_BAD_ARG;
    return run_producer(h, static_cast<cudaStream_t>(cuda_stream), 0, T, d, V, dtype, hidden, ld_hidden, W, ldw_k, ldw_v, mask, k,
                        nullptr, 0, idx_out, ld_idx, logp_out, ld_logp, lse_out);
}

extern "C" opd_status_t opd_cache_sample(opd_handle_t h, void* cuda_stream, int T, int d, int V, opd_dtype_t dtype,
    const void* hidden, long ld_hidden, const void* W, long ldw_k, long ldw_v, const unsigned char* mask, int K,
    const float* uniforms, long ld_u, int* idx_out, long ld_idx, float* logp_out, long ld_logp, float* lse_out) {
    if (!h) return OPD_ERR_BAD_ARG;
    return run_producer(h, static_cast<cudaStream_t>(cuda_stream), 1, T, d, V, dtype, hidden, ld_hidden, W, ldw_k, ldw_v, mask, K,
                        uniforms, ld_u, idx_out, ld_idx, logp_out, ld_logp, lse_out);
}

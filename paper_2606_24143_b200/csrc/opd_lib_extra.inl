// Debug / verification entry points and the host-buffer entry point.  Included by opd_lib.cu.

extern "C" opd_status_t opd_debug_logits(opd_handle_t h, void* cuda_stream, int T, int d, int V, opd_dtype_t dtype,
    const void* hidden, long ld_hidden, const void* W, long ldw_k, long ldw_v, const int* cache_idx, long ld_cache, int C,
    float* logits_out, float* gathered_out) {
    if (!h) return OPD_ERR_BAD_ARG;
    if (!logits_out) OPD_FAIL(h, OPD_ERR_BAD_ARG, "logits_out is null");
    PathIO a{};
    a.T = T; a.d = d; a.V = V; a.dtype = dtype; a.hidden = hidden; a.ld_hidden = ld_hidden; a.W = W; a.ldw_k = ldw_k; a.ldw_v = ldw_v;
    a.cache_idx = cache_idx; a.ld_cache = ld_cache; a.mode = OPD_FKL_TOPK; a.k_or_K = C;
    a.dbg_logits = logits_out; a.dbg_gathered = gathered_out; a.stop_after_fwd = true; a.all_live = true;
    return run_path(h, static_cast<cudaStream_t>(cuda_stream), a);
}

extern "C" opd_status_t opd_debug_gemm(opd_handle_t h, void* cuda_stream, int M, int N, int K, const void* A, int a_mn,
                                       const void* B, int b_mn, float* D) {
    if (!h || !A || !B || !D) return OPD_ERR_BAD_ARG;
    if (!h->arch_ok) OPD_FAIL(h, OPD_ERR_ARCH, "device %d is not compute capability 10.x", h->device);
    if (M < 1 || N < 1 || K < 1 || M % 8 || N % 8 || K % 8) OPD_FAIL(h, OPD_ERR_BAD_SHAPE, "M, N, K must be positive multiples of 8");
    if (!get_encode_fn()) OPD_FAIL(h, OPD_ERR_CUDA, "cuTensorMapEncodeTiled not available");
    OPD_ON_DEVICE(h);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    CUtensorMap tA, tB;
    bool ok = true;
    h->cg = cta_group_setting();
    if (a_mn) ok &= make_map(&tA, A, M, K, 1, (uint64_t)M * 2, (uint64_t)M * K * 2, MN_BOX);
    else      ok &= make_map(&tA, A, K, M, 1, (uint64_t)K * 2, (uint64_t)M * K * 2, BM);
    if (b_mn) ok &= make_map(&tB, B, N, K, 1, (uint64_t)N * 2, (uint64_t)N * K * 2, MN_BOX);
    else      ok &= make_map(&tB, B, K, N, 1, (uint64_t)K * 2, (uint64_t)N * K * 2, BN / h->cg);
    if (!ok) OPD_FAIL(h, OPD_ERR_CUDA, "cuTensorMapEncodeTiled failed");
    GemmParams gp{};
    gp.M = M; gp.N = N; gp.K = K; gp.num_n = ceil_div(N, BN); gp.group_m = 8;
    gp.a_mn = a_mn ? 1 : 0; gp.b_mn = b_mn ? 1 : 0;
    set_segments(gp, 1);
    gp.tok_dim = TOK_NONE; gp.n_live = nullptr;
    StoreEpi::Params ep{D, (long)N};
    h->n_kernels = h->n_gemm = 0;
    OPD_CUDA(h, launch_gemm<StoreEpi>(h, st, tA, tB, gp, ep));
    return OPD_OK;
}

// Test aid: n_ctas CTAs that each fill an SM's shared memory (one CTA per SM) and spin for `milliseconds`.  Used to check
// that the persistent backward completes while another kernel holds SMs (tests/test_robustness_gpu.py).
__global__ void __launch_bounds__(32) k_occupy(unsigned long long ns) {
    unsigned long long t0, t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    do {
        __nanosleep(2000);
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    } while (t - t0 < ns);
}
extern "C" opd_status_t opd_debug_occupy(opd_handle_t h, void* cuda_stream, int n_ctas, float milliseconds) {
    if (!h) return OPD_ERR_BAD_ARG;
    if (n_ctas < 1 || n_ctas > 1024 || !(milliseconds > 0.f) || milliseconds > 10000.f)
        OPD_FAIL(h, OPD_ERR_BAD_ARG, "n_ctas in [1,1024], milliseconds in (0, 10000]");
    OPD_ON_DEVICE(h);
    const int smem = 200 * 1024;
    OPD_CUDA(h, cudaFuncSetAttribute(k_occupy, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    k_occupy<<<n_ctas, 32, smem, static_cast<cudaStream_t>(cuda_stream)>>>(static_cast<unsigned long long>(milliseconds * 1e6));
    OPD_CUDA(h, cudaGetLastError());
    return OPD_OK;
}

// ---------------------------------------------------------------- host-buffer entry points
// Two staging slots, three streams (copy-in, compute, copy-out): a caller that alternates slots overlaps the H2D copy of
// step i+1 and the D2H copy of step i-1 with the kernels of step i.  opd_loss_fwd_bwd_host = submit + wait on slot 0.
static opd_status_t host_streams(opd_handle_s* h) {
    if (h->host_stream) return OPD_OK;
    OPD_CUDA(h, cudaStreamCreateWithFlags(&h->host_stream, cudaStreamNonBlocking));
    OPD_CUDA(h, cudaStreamCreateWithFlags(&h->host_in, cudaStreamNonBlocking));
    OPD_CUDA(h, cudaStreamCreateWithFlags(&h->host_out, cudaStreamNonBlocking));
    for (int s = 0; s < 2; ++s) {
        OPD_CUDA(h, cudaEventCreateWithFlags(&h->ev_in[s], cudaEventDisableTiming));
        OPD_CUDA(h, cudaEventCreateWithFlags(&h->ev_c[s], cudaEventDisableTiming));
        OPD_CUDA(h, cudaEventCreateWithFlags(&h->ev_out[s], cudaEventDisableTiming));
    }
    return OPD_OK;
}

extern "C" opd_status_t opd_loss_fwd_bwd_host_submit(opd_handle_t h, int slot, int T, int d, int V, opd_dtype_t dtype,
    const void* hidden_h, const void* W_h, const int* idx_h, const float* lam_h, const float* old_h, const unsigned char* mask_h,
    opd_mode_t mode, int k_or_K, unsigned flags, float norm_override,
    float* loss_h, float* ptk_h, void* gh_h, void* gw_h) {
    if (!h) return OPD_ERR_BAD_ARG;
    if (slot < 0 || slot > 1) OPD_FAIL(h, OPD_ERR_BAD_ARG, "slot must be 0 or 1");
    if (h->slot_busy[slot]) OPD_FAIL(h, OPD_ERR_BAD_ARG, "slot %d is in flight: call opd_loss_fwd_bwd_host_wait first", slot);
    if (!hidden_h || !W_h || !idx_h || !lam_h || !mask_h) OPD_FAIL(h, OPD_ERR_BAD_ARG, "null host input");
    if (flags & OPD_F_GRADW_ACCUM)
        OPD_FAIL(h, OPD_ERR_BAD_ARG, "OPD_F_GRADW_ACCUM is not available through the host entry points (grad_W is staged on the device "
                 "per call; accumulate on the host, or use opd_loss_fwd_bwd with a device grad_W)");
    int kf, Km;
    const int C = cache_width(mode, k_or_K, &kf, &Km);
    opd_status_t s = check_shape(h, T, d, V, C);
    if (s != OPD_OK) return s;
    OPD_ON_DEVICE(h);
    s = host_streams(h);
    if (s != OPD_OK) return s;
    const size_t esz = dtype == OPD_FP32 ? 4 : 2;
    const bool bwd = !(flags & OPD_F_FWD_ONLY);
    const size_t gwsz = (flags & OPD_F_GRADW_BF16) ? 2 : 4;
    size_t o = 0;
    auto take = [&](size_t b) { size_t r = o; o = align_up(o + b, 256); return r; };
    const size_t o_hid = take((size_t)T * d * esz), o_w = take((size_t)d * V * esz), o_idx = take((size_t)T * C * 4),
                 o_lam = take((size_t)T * C * 4), o_old = take((size_t)T * C * 4), o_mask = take(T), o_loss = take(4),
                 o_ptk = take((size_t)T * 4), o_gh = take(bwd ? (size_t)T * d * esz : 0), o_gw = take(bwd ? (size_t)d * V * gwsz : 0);
    if (h->stage_bytes[slot] < o) {
        if (h->stage[slot]) cudaFree(h->stage[slot]);
        h->stage[slot] = nullptr; h->stage_bytes[slot] = 0;
        cudaError_t e = cudaMalloc(&h->stage[slot], o);
        if (e != cudaSuccess) OPD_FAIL(h, OPD_ERR_WORKSPACE, "cudaMalloc(%zu) for host staging failed: %s", o, cudaGetErrorString(e));
        h->stage_bytes[slot] = o;
    }
    uint8_t* sb = static_cast<uint8_t*>(h->stage[slot]);
    size_t up = 0, down = 0;
    cudaStream_t sin = h->host_in, sc = h->host_stream, sout = h->host_out;
    auto h2d = [&](size_t off, const void* src, size_t b) { up += b; return cudaMemcpyAsync(sb + off, src, b, cudaMemcpyHostToDevice, sin); };
    OPD_CUDA(h, h2d(o_hid, hidden_h, (size_t)T * d * esz));
    OPD_CUDA(h, h2d(o_w, W_h, (size_t)d * V * esz));
    OPD_CUDA(h, h2d(o_idx, idx_h, (size_t)T * C * 4));
    OPD_CUDA(h, h2d(o_lam, lam_h, (size_t)T * C * 4));
    if (old_h) OPD_CUDA(h, h2d(o_old, old_h, (size_t)T * C * 4));
    OPD_CUDA(h, h2d(o_mask, mask_h, T));
    OPD_CUDA(h, cudaEventRecord(h->ev_in[slot], sin));
    OPD_CUDA(h, cudaStreamWaitEvent(sc, h->ev_in[slot], 0));
    s = opd_loss_fwd_bwd(h, sc, T, d, V, dtype, sb + o_hid, d, sb + o_w, V, 1, reinterpret_cast<int*>(sb + o_idx), C,
                         reinterpret_cast<float*>(sb + o_lam), old_h ? reinterpret_cast<float*>(sb + o_old) : nullptr, sb + o_mask,
                         mode, k_or_K, flags, norm_override, reinterpret_cast<float*>(sb + o_loss),
                         reinterpret_cast<float*>(sb + o_ptk), nullptr, nullptr, bwd ? sb + o_gh : nullptr, d,
                         bwd ? sb + o_gw : nullptr, V, 1);
    if (s != OPD_OK) return s;
    OPD_CUDA(h, cudaEventRecord(h->ev_c[slot], sc));
    OPD_CUDA(h, cudaStreamWaitEvent(sout, h->ev_c[slot], 0));
    auto d2h = [&](void* dst, size_t off, size_t b) { down += b; return cudaMemcpyAsync(dst, sb + off, b, cudaMemcpyDeviceToHost, sout); };
    if (loss_h) OPD_CUDA(h, d2h(loss_h, o_loss, 4));
    if (ptk_h) OPD_CUDA(h, d2h(ptk_h, o_ptk, (size_t)T * 4));
    if (bwd && gh_h) OPD_CUDA(h, d2h(gh_h, o_gh, (size_t)T * d * esz));
    if (bwd && gw_h) OPD_CUDA(h, d2h(gw_h, o_gw, (size_t)d * V * gwsz));
    OPD_CUDA(h, cudaEventRecord(h->ev_out[slot], sout));
    // the next copy-in into THIS slot must not start before these kernels have consumed it: the caller waits on the slot
    h->slot_h2d[slot] = up; h->slot_d2h[slot] = down; h->slot_busy[slot] = true;
    return OPD_OK;
}

extern "C" opd_status_t opd_loss_fwd_bwd_host_wait(opd_handle_t h, int slot, size_t* h2d_bytes, size_t* d2h_bytes) {
    if (!h) return OPD_ERR_BAD_ARG;
    if (slot < 0 || slot > 1) OPD_FAIL(h, OPD_ERR_BAD_ARG, "slot must be 0 or 1");
    if (!h->slot_busy[slot]) OPD_FAIL(h, OPD_ERR_BAD_ARG, "nothing was submitted on slot %d", slot);
    OPD_CUDA(h, cudaEventSynchronize(h->ev_out[slot]));
    h->slot_busy[slot] = false;
    if (h2d_bytes) *h2d_bytes = h->slot_h2d[slot];
    if (d2h_bytes) *d2h_bytes = h->slot_d2h[slot];
    return OPD_OK;
}

extern "C" opd_status_t opd_loss_fwd_bwd_host(opd_handle_t h, int T, int d, int V, opd_dtype_t dtype,
    const void* hidden_h, const void* W_h, const int* idx_h, const float* lam_h, const float* old_h, const unsigned char* mask_h,
    opd_mode_t mode, int k_or_K, unsigned flags, float norm_override,
    float* loss_h, float* ptk_h, void* gh_h, void* gw_h, size_t* h2d_bytes, size_t* d2h_bytes) {
    if (!h) return OPD_ERR_BAD_ARG;
    if (h->slot_busy[0]) OPD_FAIL(h, OPD_ERR_BAD_ARG, "slot 0 has a submitted call that was not waited for");
    opd_status_t s = opd_loss_fwd_bwd_host_submit(h, 0, T, d, V, dtype, hidden_h, W_h, idx_h, lam_h, old_h, mask_h, mode, k_or_K, flags,
                                                  norm_override, loss_h, ptk_h, gh_h, gw_h);
    if (s != OPD_OK) return s;
    return opd_loss_fwd_bwd_host_wait(h, 0, h2d_bytes, d2h_bytes);
}

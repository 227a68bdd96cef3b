/* opd.h — C ABI of libopd: the fused on-policy-distillation (OPD) loss on one B200 (sm_100a).
 *
 * Learner-side hot path of AsyncOPD (arxiv/paper_2606_24143; citations are PAPER.md lines):
 *   student logits z = hidden . W over the whole vocabulary, streamed tile by tile through
 *   tcgen05/TMEM and never stored (p_theta(.|s) is a policy over V);
 *   lse_t = log sum_v exp z_tv; l_tj = z_t[a_tj] - lse_t at the cached actions ("recompute
 *   log p_theta(a|s) for a in C_score(s)"); the estimators
 *     OPD_FKL_TOPK  sparse top-k teacher-weighted forward KL on the cached support
 *                   (Eq.(1) PAPER.md:57 restricted to S; renormalisers Eq.(9))
 *     OPD_RKL_MC    multi-sample Monte-Carlo reverse KL  L = -(1/m) sum_i rho_i sg(A_theta,i)
 *                   (Eq.(15)) with the advantage recomputed at learner
 *                   time A = log q - log p_theta and the unclipped ratio rho = p_theta / p_old
 *                   (Finding 2 PAPER.md:153)
 *     OPD_RKL_TOPK  sparse top-k reverse KL on a cached (stale) support, KL(p~ || q~) with both distributions
 *                   renormalised on S and S fixed during the update (App. A.1 Eq.(8)-(10));
 *                   the baseline the paper compares multi-sample MC against. Purely sparse gradient.
 *   loss = (1/N) sum over live tokens; and the backward into grad_hidden and grad_W, for which the
 *   softmax tiles are re-formed (never read back from memory).
 *
 * Conventions
 *   - Pointers are DEVICE pointers unless the name says host. The caller owns every buffer; inputs are
 *     never modified. All work is enqueued on `cuda_stream` (a cudaStream_t) and the call returns
 *     without synchronising (exception: OPD_F_VALIDATE_IDX, and the *_host entry point).
 *   - Errors are status codes; argument errors are detected on the host before any launch.
 *     opd_last_error() returns a host string describing the last failure on the handle.
 *   - No CPU fallback: on a device that is not compute capability 10.x every compute entry point
 *     returns OPD_ERR_ARCH.
 *   - One handle per host thread / stream. The handle owns its workspace unless opd_set_workspace
 *     was called.
 */
#ifndef OPD_H_
#define OPD_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct opd_handle_s* opd_handle_t;

typedef enum {
    OPD_OK = 0,
    OPD_ERR_BAD_ARG = -1,    /* null pointer, unknown mode/dtype/flag, misaligned pointer or stride */
    OPD_ERR_BAD_SHAPE = -2,  /* T,d,V,C out of the supported range (see opd_loss_fwd_bwd) */
    OPD_ERR_BAD_INDEX = -3,  /* OPD_F_VALIDATE_IDX found a cache index outside [0,V) on a live row */
    OPD_ERR_WORKSPACE = -4,  /* caller-provided workspace too small / allocation failed */
    OPD_ERR_ARCH = -5,       /* device is not sm_100 class */
    OPD_ERR_CUDA = -6        /* a CUDA runtime/driver call failed; see opd_last_error */
} opd_status_t;

typedef enum { OPD_FKL_TOPK = 0, OPD_RKL_MC = 1, OPD_MIXED = 2, OPD_RKL_TOPK = 3 } opd_mode_t;
typedef enum { OPD_BF16 = 0, OPD_FP32 = 1 } opd_dtype_t;

enum {
    OPD_F_NO_RENORM_TEACHER = 1, /* FKL: do not renormalise the cached teacher scores on S (truncated sum)      */
    OPD_F_RENORM_STUDENT = 2,    /* FKL: renormalise the student on S too (paper-literal Eq.(9); sparse backward) */
    OPD_F_GRADW_ACCUM = 4,       /* grad_W += ... instead of overwrite (micro-batches)                           */
    OPD_F_GRADW_BF16 = 8,        /* grad_W is a bf16 array: sums are kept in fp32 scratch and rounded once at the end
                                    (reading Q15: the paper does not fix the gradient dtype); +4*d*V bytes of workspace */
    OPD_F_VALIDATE_IDX = 16,     /* check cache indices of live rows; makes the call synchronous                 */
    OPD_F_FWD_ONLY = 32,         /* loss / per-token outputs only; grad pointers may be NULL                     */
    /* reverse-KL surrogate of the 2x2 ablation, Eq.(6),(7) PAPER.md:132-141 (default: A_theta, no clip = Eq.(15)) */
    OPD_F_SUR_CLIP = 64,         /* PPO clip of rho to [1-eps, 1+eps], eps = 0.2                  */
    OPD_F_SUR_A_OLD = 128,       /* frozen rollout-time advantage A_old = log q - log p_old instead of A_theta   */
    OPD_F_DENSE_REVERSE = 256    /* opd_dense_kl_fwd_bwd only: reverse direction KL(p || q), Eq.(2)  */
};

/* lifetime ------------------------------------------------------------------------------------- */
opd_status_t opd_create(opd_handle_t* out, int device);
opd_status_t opd_destroy(opd_handle_t h);
const char* opd_last_error(opd_handle_t h); /* host string, valid until the next call on h */
const char* opd_version(void);
/* ABI revision of this header. It goes up whenever an existing entry point changes its argument list (a caller built against
 * an older header would otherwise link and pass shifted arguments silently): 1 = round-1 header; 2 = opd_set_diagnostics took
 * (rows, cols), opd_cache_topk / opd_cache_sample took a mask; 3 = opd_abi_version and opd_loss_fwd_bwd_static added (no
 * signature changed). opd_abi_version() returns the value the LIBRARY was built with: compare it with OPD_ABI_VERSION once
 * after loading and refuse to run on a mismatch (paper_2606_24143_b200/opd.py does). */
#define OPD_ABI_VERSION 3
int opd_abi_version(void);

/* workspace ------------------------------------------------------------------------------------
 * Bytes of device scratch one opd_loss_fwd_bwd call with these arguments needs. No buffer of size
 * O(T*V) exists: the largest items are the compacted copy of hidden (T*d), the per-tile (max,sumexp)
 * partials (T*ceil(V/256)*8 B) and, aliased with them, a two- or three-deep ring of bounded super-tiles of re-formed softmax
 * gradients G (up to 4096 token rows x 16384 vocabulary columns of bf16 each; the planner takes the widest that keeps the
 * T-dependent scratch under 4.8% of the bf16 logits) plus fp32 grad_hidden partial sums of one token super-tile, consumed out
 * of L2 by the backward contractions (C4: 4096 x 8192 tiles, 477 MB in total, 4.8% of the bf16 logits). The modes whose gradient is purely sparse
 * (OPD_RKL_TOPK; OPD_FKL_TOPK with OPD_F_RENORM_STUDENT) instead need 16 bytes per cache entry for a column sort (their
 * grad_W is a segmented sum per column, bit-reproducible, no atomics) and, only when W is stored [d,V], a transposed copy of
 * W (2*d*V bytes for bf16; a [V,d] lm_head.weight needs none), plus 4*d bytes per 256 cache entries for the partial sums of
 * hot columns. OPD_F_GRADW_BF16 adds 4*d*V bytes (fp32 sums behind the bf16 grad_W).
 * The handle-owned workspace only grows: a call that needs more than any earlier call on the handle frees and reallocates
 * it, which synchronises the device (that one call is not asynchronous) and is refused inside a stream capture
 * (OPD_ERR_WORKSPACE: run the shapes once eagerly first, or provide the memory with opd_set_workspace). */
size_t opd_workspace_bytes(int T, int d, int V, int C, opd_dtype_t dtype, opd_mode_t mode, unsigned flags);
/* Optional: use caller memory (256-byte aligned) instead of the handle's own allocation. */
opd_status_t opd_set_workspace(opd_handle_t h, void* ws, size_t bytes);

/* the hot path --------------------------------------------------------------------------------
 * hidden   [T,d], row stride ld_hidden elements, dtype bf16 or fp32.
 * W        logical W(k,v), k in [0,d), v in [0,V): element (k,v) at W[k*ldw_k + v*ldw_v]; exactly one of
 *          the strides is 1 ([d,V] row-major: ldw_v = 1;  [V,d] row-major lm_head.weight: ldw_k = 1).
 * cache_idx [T,C] int32 in [0,V) (row stride ld_cache, also used for the two float caches);
 * cache_teacher_logp [T,C] log q(a|s); cache_old_logp [T,C] log p_old(a|s) (may be NULL for OPD_FKL_TOPK / OPD_RKL_TOPK).
 * mask     [T] bytes: 0 = masked (row contributes nothing, its cache row is never read).
 *          OPD_MIXED: 1 = FKL_TOPK row, 2 = RKL_MC row; one token-mean over all live rows.
 * k_or_K   cache width C (1..64). OPD_MIXED: k | (K << 16); FKL rows use the first k slots, MC rows the
 *          first K; C = max(k,K).
 * norm_override  > 0: divide by it instead of N = number of live tokens (N = 0 -> loss 0, grads 0).
 * loss [1], per_token_kl [T] (0 on masked rows); optional lse_out [T], student_logp_out [T,C] (row stride
 *          ld_cache; log p_theta(a_tj|s_t), written on live rows' used slots only).
 * grad_hidden [T,d] dtype of hidden, row stride ld_gh, masked rows exactly 0.
 * grad_W   fp32 (bf16 with OPD_F_GRADW_BF16), same logical layout as W: element (k,v) at grad_W[k*ldgw_k + v*ldgw_v], the
 *          unit stride must be the same one as W's. Overwritten (no need to zero it) unless OPD_F_GRADW_ACCUM.
 * Supported shapes: 1 <= T < 2^24, d % 64 == 0, 64 <= d <= 16384, V % 8 == 0, 256 <= V < 2^24, 1 <= C <= 64;
 *          hidden / W / grad bases 16-byte aligned; non-unit strides multiples of 8 (bf16) / 4 (fp32) elements.
 * Precision: bf16 inputs are used as they are, accumulation is fp32; fp32 inputs are split into three
 *          bf16 terms each (error ~2^-23 per product), so fp32 results are fp32-accurate. */
opd_status_t opd_loss_fwd_bwd(opd_handle_t h, void* cuda_stream,
    int T, int d, int V, opd_dtype_t dtype,
    const void* hidden, long ld_hidden,
    const void* W, long ldw_k, long ldw_v,
    const int* cache_idx, long ld_cache,
    const float* cache_teacher_logp,
    const float* cache_old_logp,
    const unsigned char* mask,
    opd_mode_t mode, int k_or_K,
    unsigned flags, float norm_override,
    float* loss,
    float* per_token_kl,
    float* lse_out, float* student_logp_out,
    void* grad_hidden, long ld_gh,
    void* grad_W, long ldgw_k, long ldgw_v);

/* The same call for callers that must not allocate device memory -------------------------------------------------------
 * Who this is for. opd_loss_fwd_bwd keeps its scratch in a buffer the handle obtains with cudaMalloc (and regrows with
 * cudaFree + cudaMalloc when a bigger shape arrives). Two kinds of caller cannot live with that:
 *   - a learner that shares the GPU with something that took the rest of HBM at start-up (an inference engine's KV pool, a
 *     framework's caching allocator sized to the device): a raw cudaMalloc there simply fails, or succeeds and starves the
 *     other tenant; such a caller gets all its device memory handed to it and has no spare pointer to lend as workspace;
 *   - a caller inside a latency-critical loop that keeps several streams busy: cudaMalloc / cudaFree synchronise the whole
 *     device, so one call with a new shape stalls every other stream of the process.
 * opd_loss_fwd_bwd_static takes the arguments of opd_loss_fwd_bwd, computes the same results with the same kernels, and
 * keeps ALL of its scratch in a fixed array of OPD_STATIC_SCRATCH_BYTES that is part of the library image (a file-scope
 * `static __device__` array in opd_lib.cu). It calls no cudaMalloc, cudaFree or other allocating routine, and neither reads
 * nor changes the handle's own workspace (the one opd_set_workspace / opd_loss_fwd_bwd use).
 *   Cost: every GPU on which the library's kernels are loaded holds those OPD_STATIC_SCRATCH_BYTES (32 MiB) from module load
 *     until the process exits, whether or not this entry point is ever called.
 *   Limit: the call is refused (OPD_ERR_WORKSPACE, nothing launched, opd_last_error names both numbers) when
 *     opd_workspace_bytes(T, d, V, C, dtype, mode, flags) > OPD_STATIC_SCRATCH_BYTES. That covers e.g. fp32 T=256, d=256,
 *     V=4096 (15.7 MiB), bf16 T=1024, d=1024, V=32768 with gradients (18.2 MiB), and bf16 T=4096, d=1024, V=32768 with
 *     OPD_F_FWD_ONLY (12.9 MiB); bigger problems must be cut into token chunks by the caller (OPD_F_GRADW_ACCUM + norm_override)
 *     or go through opd_loss_fwd_bwd.
 *   Set-up: the first call on each device looks up the device address of the array (cudaGetSymbolAddress, with the handle's
 *     device current; this may load the library's device code on that GPU) and remembers it; later calls only launch. Make
 *     that first call early, in ordinary eager execution, before any stream capture is begun.
 *   Sharing: there is ONE array per GPU for the whole process, shared by every handle and every stream. Each call clears the
 *     parts that must start at zero and overwrites the rest, so back-to-back calls on one stream are independent of what the
 *     previous call left behind; but two calls whose kernels can be in flight on the same GPU at the same time (different
 *     streams, different threads, different handles) race on it and both return garbage. Serialise them on one stream. */
#define OPD_STATIC_SCRATCH_BYTES (32u << 20)
opd_status_t opd_loss_fwd_bwd_static(opd_handle_t h, void* cuda_stream,
    int T, int d, int V, opd_dtype_t dtype,
    const void* hidden, long ld_hidden,
    const void* W, long ldw_k, long ldw_v,
    const int* cache_idx, long ld_cache,
    const float* cache_teacher_logp,
    const float* cache_old_logp,
    const unsigned char* mask,
    opd_mode_t mode, int k_or_K,
    unsigned flags, float norm_override,
    float* loss,
    float* per_token_kl,
    float* lse_out, float* student_logp_out,
    void* grad_hidden, long ld_gh,
    void* grad_W, long ldgw_k, long ldgw_v);

/* Same computation with HOST buffers (pinned or pageable): copies the inputs to handle-owned device
 * buffers, runs opd_loss_fwd_bwd, copies loss / per_token_kl / grad_hidden / grad_W back and
 * synchronises. All arrays are dense (ld = inner extent); W is [d,V] row-major. Pointers that are NULL
 * among the outputs are skipped. *h2d_bytes / *d2h_bytes (may be NULL) receive the bytes copied.
 * OPD_F_GRADW_BF16: grad_W_host is bf16 (halves the largest copy back). OPD_F_GRADW_ACCUM is refused (OPD_ERR_BAD_ARG): the
 * device copy of grad_W is per call. The caller's current device is left unchanged by every entry point. */
opd_status_t opd_loss_fwd_bwd_host(opd_handle_t h,
    int T, int d, int V, opd_dtype_t dtype,
    const void* hidden_host, const void* W_host,
    const int* cache_idx_host, const float* cache_teacher_logp_host, const float* cache_old_logp_host,
    const unsigned char* mask_host,
    opd_mode_t mode, int k_or_K, unsigned flags, float norm_override,
    float* loss_host, float* per_token_kl_host, void* grad_hidden_host, void* grad_W_host,
    size_t* h2d_bytes, size_t* d2h_bytes);

/* Pipelined form of the host entry point: two staging slots (0, 1) and separate copy-in / compute / copy-out streams.
 * _submit enqueues the H2D copies, the kernels and the D2H copies of one step on `slot` and returns; _wait blocks until
 * that slot's results are in the host buffers (which must stay valid, and should be pinned, until then). Alternating
 * the slots overlaps the copies of neighbouring steps with the kernels of the current one:
 *     submit(0, step 0); for i >= 1: submit(i % 2, step i); wait((i - 1) % 2);   ...  wait(last % 2)
 * A slot must be waited for before it is submitted to again (OPD_ERR_BAD_ARG otherwise). */
opd_status_t opd_loss_fwd_bwd_host_submit(opd_handle_t h, int slot,
    int T, int d, int V, opd_dtype_t dtype,
    const void* hidden_host, const void* W_host,
    const int* cache_idx_host, const float* cache_teacher_logp_host, const float* cache_old_logp_host,
    const unsigned char* mask_host,
    opd_mode_t mode, int k_or_K, unsigned flags, float norm_override,
    float* loss_host, float* per_token_kl_host, void* grad_hidden_host, void* grad_W_host);
opd_status_t opd_loss_fwd_bwd_host_wait(opd_handle_t h, int slot, size_t* h2d_bytes, size_t* d2h_bytes);

/* cache producers -------------------------------------------------------------------------------
 * The steps either side of the learner path that build the finite caches it consumes, on the same
 * streamed contraction (the logits are never stored).  hidden / W / dtype / strides as for opd_loss_fwd_bwd.  mask [T] bytes
 * (may be NULL = every row): rows with mask 0 (padding) are not scored and their rows of the outputs are not written.
 * Outputs are device arrays with row strides ld_idx / ld_logp (>= k resp. K); lse_out [T] may be NULL.
 *
 * opd_cache_topk    S_t = TopK(softmax(hidden_t . W), k), the support the scoring model selects:
 *                   idx_out [T,k] in descending order of probability (ties: lowest index first),
 *                   logp_out [T,k] the full-vocabulary-normalised log-probs on it.  1 <= k <= min(64, V).
 *                   Synchronises the stream at the end (OPD_ERR_WORKSPACE if more than max(4k,256) logits of a scored row
 *                   tie at its selection threshold, e.g. an all-zero padding row that was not masked).
 * opd_cache_sample  K draws per row from softmax(hidden_t . W), iid WITH replacement, by inverse-CDF
 *                   from the caller's uniforms u_tj in [0,1) (uniforms [T,K], row stride ld_u): a_tj is the first index v
 *                   whose cumulative probability sum_{v'<=v} p(v') reaches u_tj (cumulated in vocabulary order, fp32);
 *                   idx_out [T,K] and logp_out [T,K] = log p(a_tj) in the caller's slot order.  1 <= K <= 64.
 * opd_cache_workspace_bytes  device scratch either call needs (pass 0 for the one not used). */
size_t opd_cache_workspace_bytes(int T, int d, int V, opd_dtype_t dtype, int k_top, int K_samples);
opd_status_t opd_cache_topk(opd_handle_t h, void* cuda_stream, int T, int d, int V, opd_dtype_t dtype,
    const void* hidden, long ld_hidden, const void* W, long ldw_k, long ldw_v, const unsigned char* mask, int k,
    int* idx_out, long ld_idx, float* logp_out, long ld_logp, float* lse_out);
opd_status_t opd_cache_sample(opd_handle_t h, void* cuda_stream, int T, int d, int V, opd_dtype_t dtype,
    const void* hidden, long ld_hidden, const void* W, long ldw_k, long ldw_v, const unsigned char* mask, int K,
    const float* uniforms, long ld_u, int* idx_out, long ld_idx, float* logp_out, long ld_logp, float* lse_out);

/* dense two-head KL -------------------------------------------------------------------------------
 * Dense full-vocabulary forward KL with the teacher's distribution recomputed from TRANSMITTED TEACHER HIDDEN STATES
 * (the direction the paper names as future work; objective and gradient: Eq.(1)):
 *     q_t = softmax(teacher_hidden_t . W_T),  p_t = softmax(hidden_t . W),
 *     per_token_kl[t] = sum_v q_tv (log q_tv - log p_tv),   loss = (1/N) sum over live tokens,   dL_t/dz_tv = p_tv - q_tv.
 * Both heads are streamed tile by tile; neither set of logits is stored (bounded L2-resident rings of q and of the
 * gradient tiles only). teacher_hidden [T,dT] (row stride ld_th) and W_T (logical [dT,V], strides ldt_k / ldt_v, either
 * storage order) have the dtype of hidden / W; dT % 64 == 0. mask [T]: 0 = masked. flags: OPD_F_GRADW_ACCUM,
 * OPD_F_FWD_ONLY, OPD_F_DENSE_REVERSE. With bf16 inputs q is rounded to bf16 before use (in the loss AND the gradient,
 * consistently).
 * OPD_F_DENSE_REVERSE: the student-weighted direction (Eq.(2); gradient Eq.(3)):
 *     per_token_kl[t] = sum_v p_tv (log p_tv - log q_tv),   dL_t/dz_tv = p_tv (log p_tv - log q_tv - per_token_kl[t]);
 * log q is kept in fp32 tiles and the per-token value is formed by one more streamed pass before the gradient tiles.
 * Other arguments and outputs as for opd_loss_fwd_bwd. */
size_t opd_dense_kl_workspace_bytes(int T, int d, int dT, int V, opd_dtype_t dtype, unsigned flags);
opd_status_t opd_dense_kl_fwd_bwd(opd_handle_t h, void* cuda_stream, int T, int d, int dT, int V, opd_dtype_t dtype,
    const void* hidden, long ld_hidden, const void* W, long ldw_k, long ldw_v,
    const void* teacher_hidden, long ld_th, const void* W_T, long ldt_k, long ldt_v,
    const unsigned char* mask, unsigned flags, float norm_override,
    float* loss, float* per_token_kl, void* grad_hidden, long ld_gh, void* grad_W, long ldgw_k, long ldgw_v);

/* Optional per-token diagnostics of the MC estimator, written by the following opd_loss_fwd_bwd calls on this
 * handle (device pointers, caller-owned; pass NULLs to switch off). rows / cols: the capacity of the arrays (token rows;
 * slots per row of rho_out, <= ld_rho): a later call with T > rows or C > cols is refused (OPD_ERR_BAD_ARG), never written
 * out of bounds:
 *   rho_out [T, ld_rho]  rho_theta(a_tj) = p_theta(a_tj|s_t) / p_old(a_tj|s_t) of every cached draw of a live RKL_MC row
 *                        (caller slot order; other entries untouched) — the quantity whose p99 tail Fig. 5 reports
 *                        (PAPER.md:149-151);
 *   var1_out [T]         unbiased sample variance over the m cached draws of the one-sample estimates
 *                        -rho_j A_theta,j, i.e. the within-prefix Var(L^MC_1 | s_t) of Eq.(16);
 *                        0 on masked / non-MC rows and when m = 1. */
opd_status_t opd_set_diagnostics(opd_handle_t h, int rows, int cols, float* rho_out, long ld_rho, float* var1_out);

/* Sequence-level diagnostics of App. E (Eq.(17); Table 6, second column): "the same
 * estimator averaged over generated timesteps". cu_seqlens [n_seq + 1] (device int32): sequence n owns the token rows
 * [cu_seqlens[n], cu_seqlens[n+1]). The following OPD_RKL_MC / OPD_MIXED calls on this handle write, per sequence n
 * (device float arrays of n_seq entries, caller-owned; T_n = its live RKL_MC rows; 0 where T_n = 0):
 *   seq_mean_m[n] = (1/T_n) sum_t L^MC_m(theta; s_t)         the m-sample estimator of Eq.(15) averaged over timesteps
 *   seq_mean_1[n] = (1/T_n) sum_t L^MC_1(theta; s_t)         the same with the first cached draw of every row only
 *   seq_var_m[n]  = (1/T_n^2) sum_t Var^(L^MC_1 | s_t) / m   the variance of seq_mean_m over the local draws with the prefix
 *                   path fixed, from the within-prefix sample variances of Eq.(16) (draws are iid)
 * R_m^seq is a ratio of variances of these sequence means (m-sample over one-sample) which the caller forms over its
 * sequences or batches. Pass n_seq = 0 to switch off.
 * The three outputs describe ONE estimator, Eq.(15) with A_theta and the unclipped ratio: while the hook is on, an
 * OPD_RKL_MC / OPD_MIXED call that carries OPD_F_SUR_CLIP or OPD_F_SUR_A_OLD is refused (OPD_ERR_BAD_ARG) — its per-token
 * values would follow the surrogate while the one-sample terms and variances would not, and their ratio would compare two
 * different objectives. */
opd_status_t opd_set_seq_diagnostics(opd_handle_t h, int n_seq, const int* cu_seqlens,
                                     float* seq_mean_m, float* seq_mean_1, float* seq_var_m);

/* debugging / verification aids ----------------------------------------------------------------
 * opd_debug_logits: runs the forward contraction kernel only and dumps the fp32 logit tiles it held in
 * TMEM to logits_out [T,V] (row stride V) and the values its epilogue gathered to gathered_out [T,C]
 * (row stride C, caller slot order). Small shapes only (it writes T*V floats). All rows are treated as live. */
opd_status_t opd_debug_logits(opd_handle_t h, void* cuda_stream, int T, int d, int V, opd_dtype_t dtype,
    const void* hidden, long ld_hidden, const void* W, long ldw_k, long ldw_v,
    const int* cache_idx, long ld_cache, int C, float* logits_out, float* gathered_out);
/* opd_debug_gemm: D[M,N] (fp32, row stride N) = A . B^T through the library's tcgen05 GEMM core.
 * A is [M,K] (a_mn_major = 0) or stored as [K,M] (a_mn_major = 1); B is [N,K] or stored as [K,N]. bf16. */
opd_status_t opd_debug_gemm(opd_handle_t h, void* cuda_stream, int M, int N, int K,
    const void* A, int a_mn_major, const void* B, int b_mn_major, float* D);
/* opd_debug_occupy: enqueue a kernel of n_ctas CTAs (one per SM: each takes 200 KB of shared memory) that spin for
 * `milliseconds`. A test aid: the persistent backward kernel must complete while such a kernel holds SMs. */
opd_status_t opd_debug_occupy(opd_handle_t h, void* cuda_stream, int n_ctas, float milliseconds);
/* Launch statistics of the last opd_loss_fwd_bwd on this handle: kernels launched, GEMM-kernel launches,
 * super-tile rows/cols used by the backward. Any pointer may be NULL. */
opd_status_t opd_last_launch_stats(opd_handle_t h, int* n_kernels, int* n_gemm_kernels, int* super_rows, int* super_cols);
/* Timing hooks: if `events` (array of 2*OPD_N_PHASES cudaEvent_t, created by the caller) is set, the next
 * calls record start/stop events around each phase on the call's stream. Pass NULL to disable. */
enum { OPD_PHASE_PREP = 0, OPD_PHASE_FWD = 1, OPD_PHASE_EST = 2, OPD_PHASE_BWD = 3, OPD_N_PHASES = 4 };
opd_status_t opd_set_phase_events(opd_handle_t h, void** events);

#ifdef __cplusplus
}
#endif
#endif /* OPD_H_ */

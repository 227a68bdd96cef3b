// libopd — C ABI (include/opd.h) of the fused OPD loss for sm_100a.  Single translation unit:
//   nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -shared -Xcompiler -fPIC opd_lib.cu -o libopd.so
#include "opd_host.cuh"
#include <mutex>

using namespace opd;

#define OPD_FAIL(h, code, ...)                                   \
    do {                                                         \
        char _b[512];                                            \
        std::snprintf(_b, sizeof _b, __VA_ARGS__);               \
        if (h) (h)->err = _b;                                    \
        return (code);                                           \
    } while (0)

#define OPD_CUDA(h, expr)                                                                              \
    do {                                                                                               \
        cudaError_t _e = (expr);                                                                       \
        if (_e != cudaSuccess) OPD_FAIL(h, OPD_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(_e)); \
    } while (0)

// Makes the handle's device current for the duration of an entry point and restores the caller's device afterwards
// (a library call must not change the caller's / torch's current device in a multi-GPU process).
struct DeviceGuard {
    int prev = -1, dev = -1;
    bool ok = true;
    explicit DeviceGuard(int device) : dev(device) {
        ok = cudaGetDevice(&prev) == cudaSuccess;
        if (ok && prev != dev) ok = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() { if (prev >= 0 && prev != dev) cudaSetDevice(prev); }
};
#define OPD_ON_DEVICE(h)                                                                                       \
    DeviceGuard _device_guard((h)->device);                                                                    \
    if (!_device_guard.ok) OPD_FAIL(h, OPD_ERR_CUDA, "cannot make device %d current", (h)->device)

extern "C" const char* opd_version(void) { return "opd-b200 0.3 (sm_100a, tcgen05/TMEM/TMA)"; }
extern "C" int opd_abi_version(void) { return OPD_ABI_VERSION; }

extern "C" opd_status_t opd_create(opd_handle_t* out, int device) {
    if (!out) return OPD_ERR_BAD_ARG;
    *out = nullptr;
    opd_handle_s* h = new opd_handle_s();
    h->device = device;
    cudaDeviceProp prop;
    cudaError_t e = cudaGetDeviceProperties(&prop, device);
    if (e != cudaSuccess) { delete h; return OPD_ERR_CUDA; }
    h->num_sms = prop.multiProcessorCount;
    h->arch_ok = (prop.major == 10);
    h->l2_bytes = prop.l2CacheSize; h->l2_persist_max = prop.persistingL2CacheMaxSize; h->l2_window_max = prop.accessPolicyMaxWindowSize;
    *out = h;
    return OPD_OK;
}

extern "C" opd_status_t opd_destroy(opd_handle_t h) {
    if (!h) return OPD_ERR_BAD_ARG;
    if (h->ws_owned && h->ws) cudaFree(h->ws);
    for (int s = 0; s < 2; ++s) {
        if (h->stage[s]) cudaFree(h->stage[s]);
        if (h->ev_in[s]) { cudaEventDestroy(h->ev_in[s]); cudaEventDestroy(h->ev_c[s]); cudaEventDestroy(h->ev_out[s]); }
    }
    if (h->host_stream) { cudaStreamDestroy(h->host_stream); cudaStreamDestroy(h->host_in); cudaStreamDestroy(h->host_out); }
    delete h;
    return OPD_OK;
}

extern "C" const char* opd_last_error(opd_handle_t h) { return h ? h->err.c_str() : "null handle"; }

static opd_status_t check_shape(opd_handle_s* h, int T, int d, int V, int C) {
    if (T < 1 || T >= (1 << 24)) OPD_FAIL(h, OPD_ERR_BAD_SHAPE, "T=%d out of range [1, 2^24)", T);
    if (d < 64 || d > 16384 || d % 64) OPD_FAIL(h, OPD_ERR_BAD_SHAPE, "d=%d must be a multiple of 64 in [64,16384]", d);
    if (V < 256 || V >= (1 << 24) || V % 8) OPD_FAIL(h, OPD_ERR_BAD_SHAPE, "V=%d must be a multiple of 8 in [256, 2^24)", V);
    if (C < 1 || C > 64) OPD_FAIL(h, OPD_ERR_BAD_SHAPE, "cache width C=%d must be in [1,64]", C);
    return OPD_OK;
}

static int cache_width(opd_mode_t mode, int k_or_K, int* k, int* K) {
    if (mode == OPD_MIXED) {
        *k = k_or_K & 0xFFFF; *K = (k_or_K >> 16) & 0xFFFF;
        return *k > *K ? *k : *K;
    }
    *k = *K = k_or_K;
    return k_or_K;
}

extern "C" size_t opd_workspace_bytes(int T, int d, int V, int C, opd_dtype_t dtype, opd_mode_t mode, unsigned flags) {
    if (T < 1 || d < 64 || V < 256 || C < 1 || C > 64) return 0;
    return make_plan(T, d, V, C, dtype == OPD_FP32, flags, (int)mode).total;
}

extern "C" opd_status_t opd_set_workspace(opd_handle_t h, void* ws, size_t bytes) {
    if (!h) return OPD_ERR_BAD_ARG;
    if (ws && (reinterpret_cast<uintptr_t>(ws) & 255)) OPD_FAIL(h, OPD_ERR_BAD_ARG, "workspace must be 256-byte aligned");
    if (h->ws_owned && h->ws) cudaFree(h->ws);
    h->ws = ws; h->ws_bytes = ws ? bytes : 0; h->ws_owned = false;
    return OPD_OK;
}

// The handle-owned workspace only ever grows.  Growing it frees and reallocates device memory, which synchronises the
// device: a call whose shapes need more scratch than any earlier call on the handle is NOT asynchronous (documented in
// opd.h; opd_set_workspace avoids it).  Inside a stream capture that is impossible: OPD_ERR_WORKSPACE instead.
static opd_status_t ensure_workspace(opd_handle_s* h, size_t need, cudaStream_t st) {
    if (h->ws && h->ws_bytes >= need) return OPD_OK;
    if (h->ws && !h->ws_owned) OPD_FAIL(h, OPD_ERR_WORKSPACE, "caller workspace has %zu bytes, %zu needed", h->ws_bytes, need);
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) == cudaSuccess && cap != cudaStreamCaptureStatusNone)
        OPD_FAIL(h, OPD_ERR_WORKSPACE, "the workspace must grow to %zu bytes, which cannot happen inside a stream capture: run the "
                 "call once eagerly with these shapes, or provide memory with opd_set_workspace", need);
    if (h->ws) { cudaFree(h->ws); h->ws = nullptr; h->ws_bytes = 0; }
    cudaError_t e = cudaMalloc(&h->ws, need);
    if (e != cudaSuccess) { h->ws = nullptr; OPD_FAIL(h, OPD_ERR_WORKSPACE, "cudaMalloc(%zu) failed: %s", need, cudaGetErrorString(e)); }
    h->ws_bytes = need; h->ws_owned = true;
    return OPD_OK;
}

extern "C" opd_status_t opd_last_launch_stats(opd_handle_t h, int* nk, int* ng, int* sr, int* sc) {
    if (!h) return OPD_ERR_BAD_ARG;
    if (nk) *nk = h->n_kernels;
    if (ng) *ng = h->n_gemm;
    if (sr) *sr = h->super_rows;
    if (sc) *sc = h->super_cols;
    return OPD_OK;
}

extern "C" opd_status_t opd_set_phase_events(opd_handle_t h, void** events) {
    if (!h) return OPD_ERR_BAD_ARG;
    h->phase_events = reinterpret_cast<cudaEvent_t*>(events);
    return OPD_OK;
}

extern "C" opd_status_t opd_set_diagnostics(opd_handle_t h, int rows, int cols, float* rho_out, long ld_rho, float* var1_out) {
    if (!h) return OPD_ERR_BAD_ARG;
    if ((rho_out || var1_out) && rows < 1) OPD_FAIL(h, OPD_ERR_BAD_ARG, "rows must be the number of token rows the arrays hold");
    if (rho_out && (cols < 1 || ld_rho < cols)) OPD_FAIL(h, OPD_ERR_BAD_ARG, "rho_out needs cols >= 1 and ld_rho >= cols");
    h->diag_rho = rho_out; h->diag_ld_rho = ld_rho; h->diag_var1 = var1_out;
    h->diag_rows = (rho_out || var1_out) ? rows : 0; h->diag_cols = rho_out ? cols : 0;
    return OPD_OK;
}

extern "C" opd_status_t opd_set_seq_diagnostics(opd_handle_t h, int n_seq, const int* cu_seqlens,
                                                float* seq_mean_m, float* seq_mean_1, float* seq_var_m) {
    if (!h) return OPD_ERR_BAD_ARG;
    if (n_seq < 0 || (n_seq > 0 && (!cu_seqlens || !seq_mean_m || !seq_mean_1 || !seq_var_m)))
        OPD_FAIL(h, OPD_ERR_BAD_ARG, "n_seq > 0 needs cu_seqlens and the three output arrays");
    h->seq_n = n_seq; h->seq_cu = cu_seqlens; h->seq_mean_m = seq_mean_m; h->seq_mean_1 = seq_mean_1; h->seq_var_m = seq_var_m;
    return OPD_OK;
}

#include "opd_lib_path.inl"
#include "opd_lib_extra.inl"
#include "opd_lib_producer.inl"
#include "opd_lib_dense.inl"

// ------------------------------------------------------------------------------------------------------------------
// opd_loss_fwd_bwd_static: the hot path for callers that are not allowed to allocate device memory (include/opd.h says who
// they are: tenants of a GPU whose free memory somebody else already took, and loops that cannot afford the device-wide
// synchronisation inside cudaMalloc / cudaFree).  All scratch of the call lives in the array below, which is part of the
// library's device image: the driver places it when the module is loaded on a GPU and it stays there until the process
// ends.  One copy per GPU, shared by every handle, stream and thread of the process.
static __device__ __align__(256) unsigned char g_static_scratch[OPD_STATIC_SCRATCH_BYTES];

// In host code `g_static_scratch` is only the host-side shadow the runtime uses to identify the symbol; its value is not a
// device address and must never reach a kernel.  The address the kernels get is the one cudaGetSymbolAddress reports for
// the device that is current at the time, looked up once per device and kept here.
static constexpr int STATIC_MAX_DEVICES = 64;
static void* g_static_scratch_addr[STATIC_MAX_DEVICES] = {};
static std::mutex g_static_scratch_mu;

// Caller has made h->device current.  First call per device: resolve and remember the array's device address.
static opd_status_t static_scratch_address(opd_handle_s* h, void** out) {
    if (h->device < 0 || h->device >= STATIC_MAX_DEVICES)
        OPD_FAIL(h, OPD_ERR_BAD_ARG, "opd_loss_fwd_bwd_static supports device ordinals below %d (handle is on %d)", STATIC_MAX_DEVICES, h->device);
    std::lock_guard<std::mutex> lock(g_static_scratch_mu);
    void*& slot = g_static_scratch_addr[h->device];
    if (!slot) {
        void* p = nullptr;
        OPD_CUDA(h, cudaGetSymbolAddress(&p, g_static_scratch));
        cudaPointerAttributes at{};
        OPD_CUDA(h, cudaPointerGetAttributes(&at, p));
        if (!p || at.type != cudaMemoryTypeDevice || at.device != h->device || (reinterpret_cast<uintptr_t>(p) & 255))
            OPD_FAIL(h, OPD_ERR_CUDA, "the static scratch array did not resolve to 256-byte aligned memory of device %d", h->device);
        slot = p;
    }
    *out = slot;
    return OPD_OK;
}

extern "C" opd_status_t opd_loss_fwd_bwd_static(opd_handle_t h, void* cuda_stream, int T, int d, int V, opd_dtype_t dtype,
    const void* hidden, long ld_hidden, const void* W, long ldw_k, long ldw_v, const int* cache_idx, long ld_cache,
    const float* cache_teacher_logp, const float* cache_old_logp, const unsigned char* mask, opd_mode_t mode, int k_or_K,
    unsigned flags, float norm_override, float* loss, float* per_token_kl, float* lse_out, float* student_logp_out,
    void* grad_hidden, long ld_gh, void* grad_W, long ldgw_k, long ldgw_v) {
    if (!h) return OPD_ERR_BAD_ARG;
    if (!h->arch_ok) OPD_FAIL(h, OPD_ERR_ARCH, "device %d is not compute capability 10.x (sm_100a required, no fallback)", h->device);
    // Size check first, on the host, before anything is launched.  (Shapes, modes and dtypes the library does not support
    // at all fall through to run_path, which reports them without touching any workspace.)
    int kf, Km;
    const int C = cache_width(mode, k_or_K, &kf, &Km);
    const bool plannable = T >= 1 && T < (1 << 24) && d >= 64 && d <= 16384 && d % 64 == 0 && V >= 256 && V < (1 << 24) && V % 8 == 0 &&
                           C >= 1 && C <= 64 && (dtype == OPD_BF16 || dtype == OPD_FP32) && (int)mode >= 0 && (int)mode <= 3;
    if (plannable) {
        const size_t need = make_plan(T, d, V, C, dtype == OPD_FP32, flags, (int)mode).total;
        if (need > (size_t)OPD_STATIC_SCRATCH_BYTES)
            OPD_FAIL(h, OPD_ERR_WORKSPACE, "opd_loss_fwd_bwd_static: T=%d d=%d V=%d C=%d needs %zu bytes of scratch, the static array holds %zu "
                     "(OPD_STATIC_SCRATCH_BYTES); split the tokens into chunks or use opd_loss_fwd_bwd", T, d, V, C, need,
                     (size_t)OPD_STATIC_SCRATCH_BYTES);
    }
    OPD_ON_DEVICE(h);
    void* scratch = nullptr;
    opd_status_t s = static_scratch_address(h, &scratch);
    if (s != OPD_OK) return s;
    // Run the unchanged path with the static array standing in for the handle's workspace: marked as not owned and of
    // fixed size, so nothing below can free or grow it (a plan that did not fit would be refused, never reallocated).
    // run_path zeroes the pieces that must start at zero (bad-index flag, gathered logits, tile counters) on every call.
    void* const keep_ws = h->ws; const size_t keep_bytes = h->ws_bytes; const bool keep_owned = h->ws_owned;
    h->ws = scratch; h->ws_bytes = OPD_STATIC_SCRATCH_BYTES; h->ws_owned = false;
    PathIO a{T, d, V, dtype, hidden, ld_hidden, W, ldw_k, ldw_v, cache_idx, ld_cache, cache_teacher_logp, cache_old_logp, mask,
             mode, k_or_K, flags, norm_override, loss, per_token_kl, lse_out, student_logp_out, grad_hidden, ld_gh,
             grad_W, ldgw_k, ldgw_v, nullptr, nullptr, false, false};
    s = run_path(h, static_cast<cudaStream_t>(cuda_stream), a);
    h->ws = keep_ws; h->ws_bytes = keep_bytes; h->ws_owned = keep_owned;
    return s;
}

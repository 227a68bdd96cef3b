"""ctypes binding of libopd.so (include/opd.h).  Argument marshalling only: every step of the path
runs in the library's CUDA kernels.  torch is used for device memory and streams.

There is no CPU fallback: if the shared library is missing, or the device is not sm_100, calls raise.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, c_char_p, c_float, c_int, c_long, c_size_t, c_ubyte, c_uint, c_void_p

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libopd.so")

OPD_OK = 0
ERR_BAD_ARG, ERR_BAD_SHAPE, ERR_BAD_INDEX, ERR_WORKSPACE, ERR_ARCH, ERR_CUDA = -1, -2, -3, -4, -5, -6
FKL_TOPK, RKL_MC, MIXED, RKL_TOPK = 0, 1, 2, 3
BF16, FP32 = 0, 1
F_NO_RENORM_TEACHER, F_RENORM_STUDENT, F_GRADW_ACCUM, F_GRADW_BF16, F_VALIDATE_IDX, F_FWD_ONLY = 1, 2, 4, 8, 16, 32
F_SUR_CLIP, F_SUR_A_OLD, F_DENSE_REVERSE = 64, 128, 256
STATIC_SCRATCH_BYTES = 32 << 20          # OPD_STATIC_SCRATCH_BYTES of include/opd.h
N_PHASES = 4
PHASE_NAMES = ("prep", "fwd", "est", "bwd")

ABI_VERSION = 3                          # OPD_ABI_VERSION of include/opd.h this binding was written against

EXPORTS = ("opd_create", "opd_destroy", "opd_last_error", "opd_version", "opd_abi_version", "opd_workspace_bytes", "opd_set_workspace",
           "opd_loss_fwd_bwd", "opd_loss_fwd_bwd_static", "opd_loss_fwd_bwd_host", "opd_loss_fwd_bwd_host_submit", "opd_loss_fwd_bwd_host_wait", "opd_debug_logits", "opd_debug_gemm", "opd_last_launch_stats",
           "opd_set_phase_events", "opd_set_diagnostics", "opd_set_seq_diagnostics", "opd_debug_occupy", "opd_cache_workspace_bytes", "opd_cache_topk", "opd_cache_sample",
           "opd_dense_kl_workspace_bytes", "opd_dense_kl_fwd_bwd")

_lib = None


class OpdError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"libopd status {status}: {msg}")
        self.status = status


def load_library():
    """Load libopd.so (built in-tree by paper_2606_24143_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise OpdError(ERR_CUDA, f"{LIB_PATH} not built: run `python -m paper_2606_24143_b200.build` (no CPU fallback exists)")
    lib = ctypes.CDLL(LIB_PATH)
    if not hasattr(lib, "opd_abi_version"):
        raise OpdError(ERR_BAD_ARG, f"{LIB_PATH} predates opd_abi_version (argument lists have changed since): rebuild it")
    lib.opd_abi_version.restype = c_int
    if lib.opd_abi_version() != ABI_VERSION:
        raise OpdError(ERR_BAD_ARG, f"{LIB_PATH} was built with OPD_ABI_VERSION {lib.opd_abi_version()}, this binding expects "
                                    f"{ABI_VERSION}: rebuild with `python -m paper_2606_24143_b200.build --force`")
    lib.opd_create.argtypes = [POINTER(c_void_p), c_int]
    lib.opd_create.restype = c_int
    lib.opd_destroy.argtypes = [c_void_p]
    lib.opd_destroy.restype = c_int
    lib.opd_last_error.argtypes = [c_void_p]
    lib.opd_last_error.restype = c_char_p
    lib.opd_version.restype = c_char_p
    lib.opd_workspace_bytes.argtypes = [c_int, c_int, c_int, c_int, c_int, c_int, c_uint]
    lib.opd_workspace_bytes.restype = c_size_t
    lib.opd_set_workspace.argtypes = [c_void_p, c_void_p, c_size_t]
    lib.opd_set_workspace.restype = c_int
    lib.opd_loss_fwd_bwd.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_int,
                                     c_void_p, c_long, c_void_p, c_long, c_long, c_void_p, c_long, c_void_p, c_void_p, c_void_p,
                                     c_int, c_int, c_uint, c_float, c_void_p, c_void_p, c_void_p, c_void_p,
                                     c_void_p, c_long, c_void_p, c_long, c_long]
    lib.opd_loss_fwd_bwd.restype = c_int
    lib.opd_loss_fwd_bwd_static.argtypes = list(lib.opd_loss_fwd_bwd.argtypes)
    lib.opd_loss_fwd_bwd_static.restype = c_int
    lib.opd_loss_fwd_bwd_host.argtypes = [c_void_p, c_int, c_int, c_int, c_int, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p,
                                          c_void_p, c_int, c_int, c_uint, c_float, c_void_p, c_void_p, c_void_p, c_void_p,
                                          POINTER(c_size_t), POINTER(c_size_t)]
    lib.opd_loss_fwd_bwd_host.restype = c_int
    lib.opd_loss_fwd_bwd_host_submit.argtypes = [c_void_p, c_int, c_int, c_int, c_int, c_int, c_void_p, c_void_p, c_void_p, c_void_p,
                                                 c_void_p, c_void_p, c_int, c_int, c_uint, c_float, c_void_p, c_void_p, c_void_p, c_void_p]
    lib.opd_loss_fwd_bwd_host_submit.restype = c_int
    lib.opd_loss_fwd_bwd_host_wait.argtypes = [c_void_p, c_int, POINTER(c_size_t), POINTER(c_size_t)]
    lib.opd_loss_fwd_bwd_host_wait.restype = c_int
    lib.opd_debug_logits.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_int, c_void_p, c_long, c_void_p, c_long, c_long,
                                     c_void_p, c_long, c_int, c_void_p, c_void_p]
    lib.opd_debug_logits.restype = c_int
    lib.opd_debug_gemm.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_void_p, c_int, c_void_p, c_int, c_void_p]
    lib.opd_debug_gemm.restype = c_int
    lib.opd_last_launch_stats.argtypes = [c_void_p, POINTER(c_int), POINTER(c_int), POINTER(c_int), POINTER(c_int)]
    lib.opd_last_launch_stats.restype = c_int
    lib.opd_cache_workspace_bytes.argtypes = [c_int, c_int, c_int, c_int, c_int, c_int]
    lib.opd_cache_workspace_bytes.restype = c_size_t
    lib.opd_cache_topk.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_int, c_void_p, c_long, c_void_p, c_long, c_long, c_void_p, c_int,
                                   c_void_p, c_long, c_void_p, c_long, c_void_p]
    lib.opd_cache_topk.restype = c_int
    lib.opd_cache_sample.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_int, c_void_p, c_long, c_void_p, c_long, c_long, c_void_p, c_int,
                                     c_void_p, c_long, c_void_p, c_long, c_void_p, c_long, c_void_p]
    lib.opd_cache_sample.restype = c_int
    lib.opd_dense_kl_workspace_bytes.argtypes = [c_int, c_int, c_int, c_int, c_int, c_uint]
    lib.opd_dense_kl_workspace_bytes.restype = c_size_t
    lib.opd_dense_kl_fwd_bwd.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_int, c_int, c_void_p, c_long, c_void_p, c_long, c_long,
                                         c_void_p, c_long, c_void_p, c_long, c_long, c_void_p, c_uint, c_float,
                                         c_void_p, c_void_p, c_void_p, c_long, c_void_p, c_long, c_long]
    lib.opd_dense_kl_fwd_bwd.restype = c_int
    lib.opd_set_diagnostics.argtypes = [c_void_p, c_int, c_int, c_void_p, c_long, c_void_p]
    lib.opd_set_diagnostics.restype = c_int
    lib.opd_set_seq_diagnostics.argtypes = [c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_void_p]
    lib.opd_set_seq_diagnostics.restype = c_int
    lib.opd_debug_occupy.argtypes = [c_void_p, c_void_p, c_int, c_float]
    lib.opd_debug_occupy.restype = c_int
    lib.opd_set_phase_events.argtypes = [c_void_p, c_void_p]
    lib.opd_set_phase_events.restype = c_int
    _lib = lib
    return lib


def _ptr(t):
    return None if t is None else c_void_p(t.data_ptr())


def _dtype_code(t: torch.Tensor) -> int:
    if t.dtype == torch.bfloat16:
        return BF16
    if t.dtype == torch.float32:
        return FP32
    raise OpdError(ERR_BAD_ARG, f"unsupported dtype {t.dtype}")


def _w_strides(W: torch.Tensor, d: int):
    """W is either [d,V] (v contiguous) or a [V,d] weight passed as W.t() view / with layout='vd'."""
    if W.dim() != 2 or W.shape[0] != d:
        raise OpdError(ERR_BAD_SHAPE, f"W must be logical [d,V]; got {tuple(W.shape)} with d={d} (pass weight.t() for a [V,d] weight)")
    if W.stride(0) != 1 and W.stride(1) != 1:
        raise OpdError(ERR_BAD_ARG, f"W must be stored [d,V] or [V,d] row-major (one unit stride); strides are {tuple(W.stride())}")
    return W.stride(0), W.stride(1)


def _marshal(hidden, W, cache_idx, lam, old, mask, host: bool = False):
    """Checks what the C ABI cannot see from raw pointers (dtype, device, strides) and normalises the cheap cases:
    int64 indices -> int32, bool mask -> uint8, non-unit inner strides / unequal cache row strides -> contiguous copies.
    Everything else raises instead of being reinterpreted silently. Returns the tensors to pass on (keep them alive)."""
    if hidden.dim() != 2:
        raise OpdError(ERR_BAD_SHAPE, f"hidden must be [T,d]; got {tuple(hidden.shape)}")
    T = hidden.shape[0]
    dev = hidden.device
    if (dev.type == "cuda") == host:
        raise OpdError(ERR_BAD_ARG, f"hidden is on {dev}; this entry point takes {'host' if host else 'CUDA'} tensors")
    for name, t in (("W", W), ("cache_idx", cache_idx), ("cache_teacher_logp", lam), ("cache_old_logp", old), ("mask", mask)):
        if t is not None and t.device != dev:
            raise OpdError(ERR_BAD_ARG, f"{name} is on {t.device}, hidden on {dev}")
    if hidden.stride(1) != 1:
        hidden = hidden.contiguous()
    if cache_idx.dim() != 2 or cache_idx.shape[0] != T:
        raise OpdError(ERR_BAD_SHAPE, f"cache_idx must be [T,C]; got {tuple(cache_idx.shape)}")
    if cache_idx.dtype == torch.int64:
        cache_idx = cache_idx.to(torch.int32)
    elif cache_idx.dtype != torch.int32:
        raise OpdError(ERR_BAD_ARG, f"cache_idx must be int32 (or int64, converted); got {cache_idx.dtype}")
    for name, t in (("cache_teacher_logp", lam), ("cache_old_logp", old)):
        if t is None:
            continue
        if t.dtype != torch.float32:
            raise OpdError(ERR_BAD_ARG, f"{name} must be float32; got {t.dtype}")
        if tuple(t.shape) != tuple(cache_idx.shape):
            raise OpdError(ERR_BAD_SHAPE, f"{name} has shape {tuple(t.shape)}, cache_idx {tuple(cache_idx.shape)}")
    caches = [t for t in (cache_idx, lam, old) if t is not None]
    if any(t.stride(1) != 1 or t.stride(0) != cache_idx.stride(0) for t in caches) or (host and cache_idx.stride(0) != cache_idx.shape[1]):
        cache_idx = cache_idx.contiguous()            # the ABI takes ONE row stride for the three cache arrays
        lam = None if lam is None else lam.contiguous()
        old = None if old is None else old.contiguous()
    if mask is not None:
        if mask.dtype == torch.bool:
            mask = mask.view(torch.uint8)
        elif mask.dtype != torch.uint8:
            raise OpdError(ERR_BAD_ARG, f"mask must be uint8 (or bool); got {mask.dtype}")
        if mask.dim() != 1 or mask.shape[0] != T:
            raise OpdError(ERR_BAD_SHAPE, f"mask must be [T]; got {tuple(mask.shape)}")
        if mask.stride(0) != 1:
            mask = mask.contiguous()
    if host:                                           # the host entry points take dense arrays, W as [d,V] row-major
        hidden = hidden.contiguous()
        W = W.contiguous()
    return hidden, W, cache_idx, lam, old, mask


class Handle:
    """One libopd handle (owns its device workspace).  One per thread / stream."""

    def __init__(self, device: int | None = None):
        self.lib = load_library()
        if device is None:
            device = torch.cuda.current_device()
        self.device = device
        self._h = c_void_p()
        st = self.lib.opd_create(ctypes.byref(self._h), device)
        if st != OPD_OK:
            raise OpdError(st, "opd_create failed")
        self._events = None

    def close(self):
        if self._h:
            self.lib.opd_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st: int):
        if st != OPD_OK:
            raise OpdError(st, self.lib.opd_last_error(self._h).decode())

    def workspace_bytes(self, T, d, V, C, dtype=BF16, mode=RKL_MC, flags=0) -> int:
        return int(self.lib.opd_workspace_bytes(T, d, V, C, dtype, mode, flags))

    def launch_stats(self) -> dict:
        a, b, c, e = c_int(), c_int(), c_int(), c_int()
        self.lib.opd_last_launch_stats(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c), ctypes.byref(e))
        return dict(kernels=a.value, gemm_kernels=b.value, super_rows=c.value, super_cols=e.value)

    def set_diagnostics(self, rho_out=None, var1_out=None):
        """opd_set_diagnostics: rho_out [T,C] / var1_out [T] float32 device tensors written by the following calls."""
        for t in (rho_out, var1_out):
            if t is not None and (t.dtype != torch.float32 or not t.is_cuda or t.stride(-1) != 1):
                raise OpdError(ERR_BAD_ARG, "diagnostics outputs must be float32 CUDA tensors with a unit inner stride")
        self._diag = (rho_out, var1_out)          # keep the tensors alive
        rows = rho_out.shape[0] if rho_out is not None else (var1_out.shape[0] if var1_out is not None else 0)
        if rho_out is not None and var1_out is not None:
            rows = min(rows, var1_out.shape[0])
        self._check(self.lib.opd_set_diagnostics(self._h, rows, rho_out.shape[1] if rho_out is not None else 0, _ptr(rho_out),
                                                 rho_out.stride(0) if rho_out is not None else 0, _ptr(var1_out)))

    def set_seq_diagnostics(self, cu_seqlens=None):
        """opd_set_seq_diagnostics: cu_seqlens [n_seq+1] int32 CUDA tensor of sequence boundaries (token offsets). Returns the
        dict of float32 [n_seq] tensors (seq_mean_m, seq_mean_1, seq_var_m) the following RKL_MC / MIXED calls fill; None
        switches the hook off."""
        if cu_seqlens is None:
            self._seq = None
            self._check(self.lib.opd_set_seq_diagnostics(self._h, 0, None, None, None, None))
            return None
        if cu_seqlens.dtype != torch.int32 or not cu_seqlens.is_cuda or cu_seqlens.dim() != 1 or cu_seqlens.numel() < 2:
            raise OpdError(ERR_BAD_ARG, "cu_seqlens must be a 1-D int32 CUDA tensor with n_seq + 1 entries")
        cu = cu_seqlens.contiguous()
        n = cu.numel() - 1
        out = {k: torch.zeros(n, dtype=torch.float32, device=cu.device) for k in ("seq_mean_m", "seq_mean_1", "seq_var_m")}
        self._seq = (cu, out)
        self._check(self.lib.opd_set_seq_diagnostics(self._h, n, _ptr(cu), _ptr(out["seq_mean_m"]), _ptr(out["seq_mean_1"]),
                                                     _ptr(out["seq_var_m"])))
        return out

    def debug_occupy(self, n_ctas: int, milliseconds: float, stream=None):
        """opd_debug_occupy: keep n_ctas SMs busy for about `milliseconds` on `stream` (a test aid: one CTA per SM)."""
        s = torch.cuda.current_stream(self.device).cuda_stream if stream is None else stream
        self._check(self.lib.opd_debug_occupy(self._h, c_void_p(s), n_ctas, float(milliseconds)))

    # ------------------------------------------------------------------ phase timing
    def enable_phase_timing(self, on: bool = True):
        if on:
            self._events = [torch.cuda.Event(enable_timing=True) for _ in range(2 * N_PHASES)]
            for e in self._events:           # force creation of the underlying cudaEvent_t
                e.record()
            arr = (c_void_p * (2 * N_PHASES))(*[c_void_p(e.cuda_event) for e in self._events])
            self._event_arr = arr
            self.lib.opd_set_phase_events(self._h, ctypes.cast(arr, c_void_p))
        else:
            self._events = None
            self.lib.opd_set_phase_events(self._h, None)

    def phase_times_ms(self, events=None) -> dict:
        torch.cuda.synchronize()
        ev = self._events if events is None else events[0]
        return {PHASE_NAMES[i]: ev[2 * i].elapsed_time(ev[2 * i + 1]) for i in range(N_PHASES)}

    def new_phase_events(self):
        """A set of 2*N_PHASES timing events (and the C array of their handles) for use_phase_events."""
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * N_PHASES)]
        for e in ev:                         # force creation of the underlying cudaEvent_t
            e.record()
        return ev, (c_void_p * (2 * N_PHASES))(*[c_void_p(e.cuda_event) for e in ev])

    def use_phase_events(self, events):
        """Record the following calls' phases into `events` (from new_phase_events); None switches the hook off."""
        self._phase_set = events             # keep alive while the library holds the pointer
        self.lib.opd_set_phase_events(self._h, None if events is None else ctypes.cast(events[1], c_void_p))

    # ------------------------------------------------------------------ the hot path
    def loss_fwd_bwd(self, hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask, mode, k_or_K, flags=0,
                     norm_override=0.0, grad_hidden=None, grad_W=None, want_lse=False, want_student_logp=False, stream=None):
        """opd_loss_fwd_bwd(hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask, mode, k_or_K)
        -> dict(loss, per_token_kl, grad_hidden, grad_W[, lse, student_logp]).  All tensors live on the GPU.
        W is the logical [d,V] matrix (any of the two layouts through its strides)."""
        hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask = _marshal(hidden, W, cache_idx, cache_teacher_logp,
                                                                                  cache_old_logp, mask)
        T, d = hidden.shape
        dt = _dtype_code(hidden)
        if W.dtype != hidden.dtype:
            raise OpdError(ERR_BAD_ARG, "hidden and W must have the same dtype")
        ldk, ldv = _w_strides(W, d)
        V = W.shape[1]
        dev = hidden.device
        fwd_only = bool(flags & F_FWD_ONLY)
        gw_dtype = torch.bfloat16 if flags & F_GRADW_BF16 else torch.float32
        loss = torch.empty(1, dtype=torch.float32, device=dev)
        ptk = torch.empty(T, dtype=torch.float32, device=dev)
        lse = torch.empty(T, dtype=torch.float32, device=dev) if want_lse else None
        slp = None
        if want_student_logp:       # student_logp_out shares the caches' row stride (include/opd.h)
            slp = torch.full((T, cache_idx.stride(0)), float("nan"), dtype=torch.float32, device=dev)
        if not fwd_only:
            if grad_hidden is None:
                grad_hidden = torch.empty_like(hidden)
            elif grad_hidden.dtype != hidden.dtype or tuple(grad_hidden.shape) != (T, d) or grad_hidden.stride(1) != 1 or grad_hidden.device != dev:
                raise OpdError(ERR_BAD_ARG, "grad_hidden must be a [T,d] tensor of hidden's dtype and device with a unit inner stride")
            if grad_W is None:
                if flags & F_GRADW_ACCUM:
                    raise OpdError(ERR_BAD_ARG, "OPD_F_GRADW_ACCUM accumulates into the caller's grad_W: pass it")
                grad_W = torch.empty_strided(tuple(W.shape), (ldk, ldv), dtype=gw_dtype, device=dev)
            elif grad_W.dtype != gw_dtype or tuple(grad_W.shape) != (d, V) or grad_W.device != dev:
                raise OpdError(ERR_BAD_ARG, f"grad_W must be a logical [d,V] {gw_dtype} tensor on {dev}")
        s = torch.cuda.current_stream(dev).cuda_stream if stream is None else stream
        gk, gv = (grad_W.stride(0), grad_W.stride(1)) if grad_W is not None else (0, 0)
        st = self.lib.opd_loss_fwd_bwd(
            self._h, c_void_p(s), T, d, V, dt, _ptr(hidden), hidden.stride(0), _ptr(W), ldk, ldv,
            _ptr(cache_idx), cache_idx.stride(0), _ptr(cache_teacher_logp), _ptr(cache_old_logp), _ptr(mask),
            mode, k_or_K, flags, float(norm_override), _ptr(loss), _ptr(ptk), _ptr(lse), _ptr(slp),
            _ptr(grad_hidden), grad_hidden.stride(0) if grad_hidden is not None else 0, _ptr(grad_W), gk, gv)
        self._check(st)
        if slp is not None:
            slp = slp[:, :cache_idx.shape[1]]
        return dict(loss=loss, per_token_kl=ptk, grad_hidden=grad_hidden, grad_W=grad_W, lse=lse, student_logp=slp)

    def loss_fwd_bwd_static(self, hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask, mode, k_or_K, out, flags=0,
                            norm_override=0.0, stream=None):
        """opd_loss_fwd_bwd_static: the same computation as loss_fwd_bwd for a caller that may not allocate GPU memory -- a
        learner whose GPU's free memory already belongs to another tenant (an inference engine's pool, a caching allocator
        sized to the device), or a loop that cannot take the device-wide stall of cudaMalloc / cudaFree.  The library keeps
        the call's scratch in a fixed 32 MiB array inside its own device image (STATIC_SCRATCH_BYTES) and this wrapper
        allocates nothing either, so the caller supplies every buffer:
          out = dict(loss [1] f32, per_token_kl [T] f32, grad_hidden [T,d] like hidden, grad_W logical [d,V] f32 (bf16 with
                     F_GRADW_BF16) with W's unit stride; optional lse [T] f32, student_logp [T, row stride of cache_idx] f32);
                grad_hidden / grad_W may be left out with F_FWD_ONLY.  The results are written into these tensors; `out` is returned.
        Inputs must already be in the form the C ABI takes (int32 indices, uint8 / bool mask, unit inner strides, one common
        row stride for the three cache arrays): where loss_fwd_bwd would make a converted copy, this raises instead.
        Raises OpdError(ERR_WORKSPACE) when the shape needs more scratch than the array holds (see workspace_bytes).
        The first call on a device resolves the array's address; make it once before any stream capture.  One array per GPU
        is shared by all handles and streams: calls that could overlap on the GPU must be serialised by the caller."""
        given = (hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask)
        ready = _marshal(*given)
        for name, a, b in zip(("hidden", "W", "cache_idx", "cache_teacher_logp", "cache_old_logp", "mask"), given, ready):
            if (a is None) != (b is None) or (a is not None and (a.data_ptr() != b.data_ptr() or a.stride() != b.stride())):
                raise OpdError(ERR_BAD_ARG, f"{name} would need a converted copy (dtype / strides); the static entry point allocates nothing")
        hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask = ready
        T, d = hidden.shape
        dt = _dtype_code(hidden)
        if W.dtype != hidden.dtype:
            raise OpdError(ERR_BAD_ARG, "hidden and W must have the same dtype")
        ldk, ldv = _w_strides(W, d)
        V = W.shape[1]
        dev = hidden.device
        fwd_only = bool(flags & F_FWD_ONLY)
        gw_dtype = torch.bfloat16 if flags & F_GRADW_BF16 else torch.float32
        want = [("loss", (1,), torch.float32), ("per_token_kl", (T,), torch.float32)]
        if not fwd_only:
            want += [("grad_hidden", (T, d), hidden.dtype), ("grad_W", (d, V), gw_dtype)]
        for name, shape, dtype in want:
            t = out.get(name)
            if t is None or t.dtype != dtype or tuple(t.shape) != shape or t.device != dev:
                raise OpdError(ERR_BAD_ARG, f"out['{name}'] must be a {shape} {dtype} tensor on {dev}")
        lse, slp = out.get("lse"), out.get("student_logp")
        if lse is not None and (lse.dtype != torch.float32 or tuple(lse.shape) != (T,) or lse.device != dev or lse.stride(0) != 1):
            raise OpdError(ERR_BAD_ARG, "out['lse'] must be a dense [T] float32 tensor on hidden's device")
        if slp is not None and (slp.dtype != torch.float32 or slp.dim() != 2 or slp.shape[0] != T or slp.device != dev or
                                slp.stride(1) != 1 or slp.stride(0) != cache_idx.stride(0)):
            raise OpdError(ERR_BAD_ARG, "out['student_logp'] must be float32 [T, .] with the row stride of cache_idx")
        gh, gw = (None, None) if fwd_only else (out["grad_hidden"], out["grad_W"])
        if gh is not None and gh.stride(1) != 1:
            raise OpdError(ERR_BAD_ARG, "out['grad_hidden'] needs a unit inner stride")
        if not (out["loss"].is_contiguous() and out["per_token_kl"].is_contiguous()):
            raise OpdError(ERR_BAD_ARG, "out['loss'] / out['per_token_kl'] must be dense")
        s = torch.cuda.current_stream(dev).cuda_stream if stream is None else stream
        gk, gv = (gw.stride(0), gw.stride(1)) if gw is not None else (0, 0)
        self._check(self.lib.opd_loss_fwd_bwd_static(
            self._h, c_void_p(s), T, d, V, dt, _ptr(hidden), hidden.stride(0), _ptr(W), ldk, ldv,
            _ptr(cache_idx), cache_idx.stride(0), _ptr(cache_teacher_logp), _ptr(cache_old_logp), _ptr(mask),
            mode, k_or_K, flags, float(norm_override), _ptr(out["loss"]), _ptr(out["per_token_kl"]), _ptr(lse), _ptr(slp),
            _ptr(gh), gh.stride(0) if gh is not None else 0, _ptr(gw), gk, gv))
        return out

    def loss_fwd_bwd_host(self, hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask, mode, k_or_K, flags=0,
                          norm_override=0.0, out=None):
        """Same call with HOST tensors (pinned or pageable, dense); copies in, runs, copies out, synchronises.
        `out`: optional dict of preallocated host tensors (loss, per_token_kl, grad_hidden, grad_W)."""
        hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask = _marshal(hidden, W, cache_idx, cache_teacher_logp,
                                                                                  cache_old_logp, mask, host=True)
        T, d = hidden.shape
        V = W.shape[1]
        dt = _dtype_code(hidden)
        fwd_only = bool(flags & F_FWD_ONLY)
        if out is None:
            out = dict(loss=torch.empty(1, dtype=torch.float32), per_token_kl=torch.empty(T, dtype=torch.float32),
                       grad_hidden=None if fwd_only else torch.empty_like(hidden),
                       grad_W=None if fwd_only else torch.empty(d, V, dtype=torch.bfloat16 if flags & F_GRADW_BF16 else torch.float32))
        up, down = c_size_t(), c_size_t()
        st = self.lib.opd_loss_fwd_bwd_host(
            self._h, T, d, V, dt, _ptr(hidden), _ptr(W), _ptr(cache_idx), _ptr(cache_teacher_logp), _ptr(cache_old_logp),
            _ptr(mask), mode, k_or_K, flags, float(norm_override), _ptr(out["loss"]), _ptr(out["per_token_kl"]),
            _ptr(out.get("grad_hidden")), _ptr(out.get("grad_W")), ctypes.byref(up), ctypes.byref(down))
        self._check(st)
        out["h2d_bytes"], out["d2h_bytes"] = up.value, down.value
        return out

    def host_submit(self, slot, hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask, mode, k_or_K, out, flags=0,
                    norm_override=0.0):
        """opd_loss_fwd_bwd_host_submit: enqueue one step on staging slot 0/1 (host tensors; `out` = dict of host tensors
        loss, per_token_kl, grad_hidden, grad_W that receive the results once host_wait(slot) has returned)."""
        hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask = _marshal(hidden, W, cache_idx, cache_teacher_logp,
                                                                                  cache_old_logp, mask, host=True)
        T, d = hidden.shape
        V = W.shape[1]
        self._pending = getattr(self, "_pending", {})
        self._pending[slot] = (hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask, out)     # keep alive
        self._check(self.lib.opd_loss_fwd_bwd_host_submit(
            self._h, slot, T, d, V, _dtype_code(hidden), _ptr(hidden), _ptr(W), _ptr(cache_idx), _ptr(cache_teacher_logp),
            _ptr(cache_old_logp), _ptr(mask), mode, k_or_K, flags, float(norm_override), _ptr(out["loss"]),
            _ptr(out["per_token_kl"]), _ptr(out.get("grad_hidden")), _ptr(out.get("grad_W"))))

    def host_wait(self, slot):
        """opd_loss_fwd_bwd_host_wait -> (out dict of the step submitted on `slot`, h2d bytes, d2h bytes)."""
        up, down = c_size_t(), c_size_t()
        self._check(self.lib.opd_loss_fwd_bwd_host_wait(self._h, slot, ctypes.byref(up), ctypes.byref(down)))
        out = self._pending.pop(slot)[-1]
        return out, up.value, down.value

    # ------------------------------------------------------------------ cache producers
    @staticmethod
    def _producer_args(hidden, W, mask):
        if hidden.dim() != 2 or not hidden.is_cuda or hidden.stride(1) != 1:
            raise OpdError(ERR_BAD_ARG, "hidden must be a [T,d] CUDA tensor with a unit inner stride")
        if W.dtype != hidden.dtype or W.device != hidden.device:
            raise OpdError(ERR_BAD_ARG, "hidden and W must have the same dtype and device")
        if mask is not None:
            if mask.dtype == torch.bool:
                mask = mask.view(torch.uint8)
            if mask.dtype != torch.uint8 or mask.dim() != 1 or mask.shape[0] != hidden.shape[0] or mask.device != hidden.device:
                raise OpdError(ERR_BAD_ARG, "mask must be a [T] uint8 / bool tensor on hidden's device")
            mask = mask.contiguous()
        return mask

    def cache_topk(self, hidden, W, k, mask=None):
        """opd_cache_topk -> (idx [T,k] int32, logp [T,k] float32, lse [T] float32): the scoring model's top-k support.
        Rows with mask == 0 are not scored (idx -1, logp -inf, lse 0 there)."""
        mask = self._producer_args(hidden, W, mask)
        T, d = hidden.shape
        V = W.shape[1]
        ldk, ldv = _w_strides(W, d)
        dev = hidden.device
        idx = torch.full((T, k), -1, dtype=torch.int32, device=dev)
        logp = torch.full((T, k), float("-inf"), dtype=torch.float32, device=dev)
        lse = torch.zeros(T, dtype=torch.float32, device=dev)
        s = torch.cuda.current_stream(dev).cuda_stream
        self._check(self.lib.opd_cache_topk(self._h, c_void_p(s), T, d, V, _dtype_code(hidden), _ptr(hidden), hidden.stride(0), _ptr(W),
                                            ldk, ldv, _ptr(mask), k, _ptr(idx), k, _ptr(logp), k, _ptr(lse)))
        return idx, logp, lse

    def cache_sample(self, hidden, W, uniforms, mask=None):
        """opd_cache_sample -> (idx [T,K] int32, logp [T,K] float32, lse [T]): K inverse-CDF draws per row from
        softmax(hidden . W) for the uniforms [T,K] (float32, in [0,1)). Rows with mask == 0 are not scored."""
        mask = self._producer_args(hidden, W, mask)
        T, d = hidden.shape
        V = W.shape[1]
        if uniforms.dtype != torch.float32 or tuple(uniforms.shape[:1]) != (T,) or uniforms.stride(1) != 1 or uniforms.device != hidden.device:
            raise OpdError(ERR_BAD_ARG, "uniforms must be a [T,K] float32 tensor on hidden's device with a unit inner stride")
        K = uniforms.shape[1]
        ldk, ldv = _w_strides(W, d)
        dev = hidden.device
        idx = torch.full((T, K), -1, dtype=torch.int32, device=dev)
        logp = torch.full((T, K), float("-inf"), dtype=torch.float32, device=dev)
        lse = torch.zeros(T, dtype=torch.float32, device=dev)
        s = torch.cuda.current_stream(dev).cuda_stream
        self._check(self.lib.opd_cache_sample(self._h, c_void_p(s), T, d, V, _dtype_code(hidden), _ptr(hidden), hidden.stride(0), _ptr(W),
                                              ldk, ldv, _ptr(mask), K, _ptr(uniforms), uniforms.stride(0), _ptr(idx), K, _ptr(logp), K, _ptr(lse)))
        return idx, logp, lse

    # ------------------------------------------------------------------ dense two-head KL
    def dense_kl_fwd_bwd(self, hidden, W, teacher_hidden, W_T, mask, flags=0, norm_override=0.0, grad_hidden=None, grad_W=None):
        """opd_dense_kl_fwd_bwd -> dict(loss, per_token_kl, grad_hidden, grad_W): dense forward KL(q || p) with
        q = softmax(teacher_hidden . W_T), p = softmax(hidden . W); W / W_T are the logical [d,V] / [dT,V] heads."""
        T, d = hidden.shape
        dT = teacher_hidden.shape[1]
        V = W.shape[1]
        ldk, ldv = _w_strides(W, d)
        tk, tv = _w_strides(W_T, dT)
        dev = hidden.device
        fwd_only = bool(flags & F_FWD_ONLY)
        loss = torch.empty(1, dtype=torch.float32, device=dev)
        ptk = torch.empty(T, dtype=torch.float32, device=dev)
        if not fwd_only:
            if grad_hidden is None:
                grad_hidden = torch.empty_like(hidden)
            if grad_W is None:
                grad_W = torch.empty_strided(tuple(W.shape), (ldk, ldv), dtype=torch.float32, device=dev)
        gk, gv = (grad_W.stride(0), grad_W.stride(1)) if grad_W is not None else (0, 0)
        s = torch.cuda.current_stream(dev).cuda_stream
        self._check(self.lib.opd_dense_kl_fwd_bwd(
            self._h, c_void_p(s), T, d, dT, V, _dtype_code(hidden), _ptr(hidden), hidden.stride(0), _ptr(W), ldk, ldv,
            _ptr(teacher_hidden), teacher_hidden.stride(0), _ptr(W_T), tk, tv, _ptr(mask), flags, float(norm_override),
            _ptr(loss), _ptr(ptk), _ptr(grad_hidden), grad_hidden.stride(0) if grad_hidden is not None else 0, _ptr(grad_W), gk, gv))
        return dict(loss=loss, per_token_kl=ptk, grad_hidden=grad_hidden, grad_W=grad_W)

    # ------------------------------------------------------------------ debug entries
    def debug_logits(self, hidden, W, cache_idx):
        T, d = hidden.shape
        V = W.shape[1]
        ldk, ldv = _w_strides(W, d)
        C = cache_idx.shape[1]
        logits = torch.empty(T, V, dtype=torch.float32, device=hidden.device)
        gathered = torch.empty(T, C, dtype=torch.float32, device=hidden.device)
        s = torch.cuda.current_stream(hidden.device).cuda_stream
        st = self.lib.opd_debug_logits(self._h, c_void_p(s), T, d, V, _dtype_code(hidden), _ptr(hidden), hidden.stride(0), _ptr(W),
                                       ldk, ldv, _ptr(cache_idx), cache_idx.stride(0), C, _ptr(logits), _ptr(gathered))
        self._check(st)
        return logits, gathered

    def debug_gemm(self, A, B, a_mn_major=False, b_mn_major=False):
        """D = A_logical[M,K] @ B_logical[N,K]^T (fp32).  A is stored [M,K] (or [K,M] if a_mn_major), same for B."""
        if a_mn_major:
            K, M = A.shape
        else:
            M, K = A.shape
        N = B.shape[1] if b_mn_major else B.shape[0]
        D = torch.empty(M, N, dtype=torch.float32, device=A.device)
        s = torch.cuda.current_stream(A.device).cuda_stream
        st = self.lib.opd_debug_gemm(self._h, c_void_p(s), M, N, K, _ptr(A), int(a_mn_major), _ptr(B), int(b_mn_major), _ptr(D))
        self._check(st)
        return D


_default = {}


def default_handle(device: int | None = None) -> Handle:
    if device is None:
        device = torch.cuda.current_device()
    if device not in _default:
        _default[device] = Handle(device)
    return _default[device]


def opd_loss_fwd_bwd(hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask, mode, k_or_K, **kw):
    """Module-level convenience: the north-star signature on the default handle of the current device."""
    return default_handle(hidden.device.index).loss_fwd_bwd(hidden, W, cache_idx, cache_teacher_logp, cache_old_logp,
                                                            mask, mode, k_or_K, **kw)

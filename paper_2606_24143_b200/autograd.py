"""torch.autograd entry to the fused OPD loss: a drop-in for a PyTorch learner (PAPER.md:334 trains with PyTorch FSDP).

    loss = opd_loss(hidden, lm_head_weight.t(), cache_idx, cache_teacher_logp, cache_old_logp, mask, RKL_MC, K)
    loss.backward()        # hidden.grad / lm_head_weight.grad come from the library's fused backward

Marshalling only: forward calls opd_loss_fwd_bwd once (loss AND both gradients are produced by that call, the
logits are never materialised); backward hands the stored gradients to autograd, scaled (out of place: a second
backward with retain_graph=True sees the same saved tensors) by the incoming scalar gradient.  Peak memory: for a bf16 head
the library is asked for a bf16 grad_W (OPD_F_GRADW_BF16: fp32 sums stay in the handle's workspace and are rounded once), so
what is saved for backward is already in the parameter's dtype (2*d*V bytes instead of 4*d*V), and the scale by the incoming
gradient writes straight into one tensor of that dtype (no fp32 temporary, no separate cast copy).
There is no PyTorch fallback: without libopd.so / off sm_100 the call raises.
"""
from __future__ import annotations

import torch

from . import opd


class _OpdLoss(torch.autograd.Function):
    @staticmethod
    def forward(ctx, hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask, mode, k_or_K, flags, norm_override):
        need_grad = hidden.requires_grad or W.requires_grad
        h = opd.default_handle(hidden.device.index)
        if need_grad and W.dtype == torch.bfloat16 and not (flags & opd.F_GRADW_ACCUM):
            flags |= opd.F_GRADW_BF16                   # the gradient autograd wants has W's dtype anyway: save it as such
        r = h.loss_fwd_bwd(hidden.detach(), W.detach(), cache_idx, cache_teacher_logp, cache_old_logp, mask, mode, k_or_K,
                           flags=flags | (0 if need_grad else opd.F_FWD_ONLY), norm_override=norm_override)
        ctx.need_grad = need_grad
        if need_grad:
            ctx.save_for_backward(r["grad_hidden"], r["grad_W"])
        ctx.w_dtype = W.dtype
        ctx.mark_non_differentiable(r["per_token_kl"])
        return r["loss"].reshape(()), r["per_token_kl"]

    @staticmethod
    def backward(ctx, g_loss, _g_ptk):
        if not ctx.need_grad:
            return (None,) * 10
        gh, gw = ctx.saved_tensors
        if g_loss is not None:                  # chain rule with the incoming scalar: out of place, without a host sync
            gh = gh * g_loss.to(gh.dtype)
            # one output in W's dtype; the product is formed in fp32 and rounded on the way out (no full-size temporary)
            gw = torch.mul(gw, g_loss.float(), out=torch.empty_like(gw, dtype=ctx.w_dtype))
        elif gw.dtype != ctx.w_dtype:
            gw = gw.to(ctx.w_dtype)
        return gh, gw, None, None, None, None, None, None, None, None


def opd_loss(hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask, mode, k_or_K, flags: int = 0,
             norm_override: float = 0.0, return_per_token: bool = False):
    """Fused OPD loss with autograd support. `W` is the logical [d,V] head (pass `lm_head.weight.t()` for a [V,d]
    parameter: the transposed view is used in place). Returns the scalar loss (and the per-token estimates)."""
    loss, ptk = _OpdLoss.apply(hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask, mode, k_or_K, flags, norm_override)
    return (loss, ptk) if return_per_token else loss
